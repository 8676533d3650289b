// dt_tiles.cu -- hits-first scheduling with a tiled image cache for surveys that do not fit HBM
// (SURVEY.md 8(f) NEXT-2).  The paper keeps its images on node-local SSD "in smaller two-dimensional blocks"
// so that "the pixels we need to gather from an image [are] more likely to be on a small number of memory
// pages", only looks pixels up AFTER the GPU has found and compacted the intersections
// (Algorithm 1), and names pipelining the two phases as future work
// (PAPER.md:330-332).  Here the images sit in page-locked host memory and the same idea becomes:
//
//   1. kernel 1 runs first -- it needs no image -- and leaves the unit's compacted hit list;
//   2. k_tile_count walks the hit entries FLAT (an entry names its exposure, dt_common.cuh) and counts the hits
//      per (exposure, 64 x 64-pixel tile);
//   3. k_tile_assign gives every tile with at least `min_hits` hits that is not resident yet a slot of the
//      device tile cache (one integer atomic per new tile) and queues it;
//   4. k_tile_fetch copies the queued tiles -- and only those -- from the device-mapped host planes into their
//      slots, 256-B row segments, coalesced, many in flight: the 2-D tiled layout is built on the way in;
//   5. kernel 3 reads a hit's pixel from its tile's slot, or, for a tile without a slot (too few hits to be
//      worth 16 KB of transfer, or the cache is full), straight from the host plane (zero-copy).
//
// The cache lives for one exposure unit (<= 512 exposures) and is shared by all orbit units of that range, so a
// tile crosses PCIe at most once per pass.  Nothing is synchronised with the host; the same pixels enter the same
// arithmetic in the same order, so results are bit-identical to the resident and the streamed runs.
#include "dt_common.cuh"
#include "dt_gather.cuh"

namespace dt {

constexpr int kTileThreads = 256;

// ---- 2: hits per (exposure, tile) -- one warp per (warp-tile of orbits, group) block, entries read flat ----
__global__ void __launch_bounds__(kTileThreads) k_tile_count(const TileParams t)
{
    const int lane = threadIdx.x & 31;
    const int64_t n_tiles = t.n_pad >> 5;
    const int64_t w = ((int64_t)blockIdx.x * kTileThreads + threadIdx.x) >> 5;       // (group, warp-tile) index
    if (w >= n_tiles * t.n_groups) return;
    const int64_t g = w / n_tiles, wt = w - g * n_tiles;
    const uint32_t bits = t.mask[g * t.n_pad + wt * 32 + lane];
    const int m = __reduce_add_sync(0xffffffffu, __popc(bits));
    if (m == 0) return;
    const uint32_t blk0 = (uint32_t)t.base[g * n_tiles + wt];
    for (int k = lane; k < m; k += 32) {
        if (!DT_IN_BOUNDS((int64_t)blk0 + k < t.offsets_cap, t.bounds)) continue;
        const uint32_t e = t.offsets[blk0 + k];
        const uint32_t off = e & kOffsetMask;
        if (!DT_IN_BOUNDS((int64_t)off < (int64_t)t.width * t.height && g * kGroup + (e >> kOffsetBits) < (uint32_t)t.n_exp, t.bounds))
            continue;
        const int y = (int)(off / (uint32_t)t.width), x = (int)(off - (uint32_t)y * (uint32_t)t.width);
        const int tile = (y >> t.ts_log2) * t.tiles_x + (x >> t.ts_log2);
        const int64_t row = g * kGroup + (e >> kOffsetBits);                         // exposure within the unit
        atomicAdd(t.tile_count + row * t.tiles_per_plane + tile, 1);
    }
}

// ---- 3: slots for the tiles worth fetching; the counts are cleared for the next orbit unit ----
__global__ void __launch_bounds__(kTileThreads) k_tile_assign(const TileParams t)
{
    const int64_t i = (int64_t)blockIdx.x * kTileThreads + threadIdx.x;
    if (i >= (int64_t)t.n_exp * t.tiles_per_plane) return;
    const int c = t.tile_count[i];
    if (c == 0) return;
    t.tile_count[i] = 0;
    if (c < t.min_hits || t.tile_slot[i] >= 0) return;
    const unsigned s = atomicAdd(t.alloc + 0, 1u);
    if (s >= (unsigned)t.capacity) return;               // cache full: this tile stays zero-copy
    t.tile_slot[i] = (int32_t)s;
    const unsigned q = atomicAdd(t.alloc + 1, 1u);
    if (DT_IN_BOUNDS(q < (unsigned)t.capacity, t.bounds)) t.fetch_list[q] = make_uint2((unsigned)i, s);
}

// ---- 4: host plane -> tile slot.  One CTA per queued tile (grid-stride), 64 threads per 256-B row segment ----
__global__ void __launch_bounds__(kTileThreads) k_tile_fetch(const TileParams t)
{
    const unsigned n = t.alloc[1];
    const int ts = 1 << t.ts_log2;
    for (unsigned q = blockIdx.x; q < n; q += gridDim.x) {
        const uint2 it = t.fetch_list[q];
        const int row = (int)(it.x / (unsigned)t.tiles_per_plane), tile = (int)(it.x - (unsigned)row * (unsigned)t.tiles_per_plane);
        const int ty = tile / t.tiles_x, tx = tile - ty * t.tiles_x;
        const int64_t j = (int64_t)t.first_exposure + row;                          // absolute exposure
        const float *src_f = t.flux_ptrs[j];
        const float *src_v = t.var_ptrs ? t.var_ptrs[j] : nullptr;
        float *dst = t.tile_buf + (int64_t)it.y * t.slot_floats;
        for (int k = threadIdx.x; k < ts * ts; k += kTileThreads) {
            const int yy = (ty << t.ts_log2) + (k >> t.ts_log2), xx = (tx << t.ts_log2) + (k & (ts - 1));
            float f = 0.f, v = 0.f;
            if (yy < t.height && xx < t.width) {
                const int64_t a = (int64_t)yy * t.width + xx;
                f = __ldcs(src_f + a);
                if (src_v) v = __ldcs(src_v + a);
            }
            dst[k] = f;
            if (src_v) dst[ts * ts + k] = v;
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(t.alloc + 2, n);              // statistics: tiles fetched
}

cudaError_t launch_tiles(const TileParams &t, int sm_count, cudaStream_t stream)
{
    if (t.n_pad <= 0 || t.n_groups <= 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(t.alloc + 1, 0, sizeof(unsigned int), stream);   // fetch queue of this unit
    if (e != cudaSuccess) return e;
    const int64_t warps = (t.n_pad >> 5) * t.n_groups;
    k_tile_count<<<(unsigned)((warps * 32 + kTileThreads - 1) / kTileThreads), kTileThreads, 0, stream>>>(t);
    const int64_t cells = (int64_t)t.n_exp * t.tiles_per_plane;
    k_tile_assign<<<(unsigned)((cells + kTileThreads - 1) / kTileThreads), kTileThreads, 0, stream>>>(t);
    k_tile_fetch<<<(unsigned)(sm_count * 8), kTileThreads, 0, stream>>>(t);
    return cudaGetLastError();
}

}  // namespace dt
