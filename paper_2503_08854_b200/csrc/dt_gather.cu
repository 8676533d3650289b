// dt_gather.cu -- kernel 3: gather + stack (sparse schedule, launcher) and the SNR finalisation.
//
// Hot-path steps 8-9 of DESIGN.md (Algorithm 1 `FindLocalSignal` + the per-orbit combination,
// PAPER.md:171-172, 182 "jointly combining the signal from all intersections").  The paper pulls
// pixels on the CPU from mmap'd SSD files; here the images are in HBM.
//
// Two schedules share the hit-list format (dtrack.h, dt_gather_hits: per (warp-tile, group) block the
// pixel offsets are exposure-major, then lane-ascending) and the per-orbit arithmetic; each launch
// enqueues both kernels and each kernel returns at once unless the unit's hit density, read on the
// device from kernel 1's counter, is in its regime (no host synchronisation between the kernels):
//   * k_gather_sparse (this file): one orbit per lane, one warp-tile per warp, many CTAs.  Per block
//     the warp transposes its 32 per-orbit masks into 32 per-exposure column masks (32 ballots) and
//     scans their popcounts; entry (lane, jj) sits at block start + prefix[jj] + popc(column[jj] &
//     lanes below).  Every lane then walks ITS OWN hits in ascending exposure order, four in
//     flight, so all lanes stay busy however few exposures a block touches.  Bound: the rate of
//     random DRAM accesses (no reuse to exploit when hits are sparse).
//     In streaming mode with few hits it can also read the pixels straight from the page-locked host
//     planes (zero-copy), so that a survey larger than HBM need not be streamed at all.
//   * k_gather_dense (dt_gather_dense.cu): one persistent wave sweeping the exposures in lock-step so
//     that the planes being gathered from stay L2-resident while every orbit of the unit reads them.
// Both accumulate S += f/v, Wt += 1/v per orbit in ascending exposure order in a lane-private
// accumulator (registers here, shared memory in the dense kernel) -- no atomics, and bit-identical
// to a sequential evaluation of the definition.
#include <math.h>

#include <algorithm>

#include "dt_common.cuh"
#include "dt_gather.cuh"

namespace dt {

constexpr int kSparseThreads = 256;

// Tiled image cache (dt_tiles.cu): the pixel (exposure j, offset a) from its tile's slot when the tile is resident.
template <bool PLANE_VAR>
__device__ __forceinline__ bool load_pixel_tiled(const GatherParams &p, int64_t j, uint32_t a, float &f, float &v)
{
    const uint32_t y = a / (uint32_t)p.width, x = a - y * (uint32_t)p.width;
    const int tile = (int)(y >> p.ts_log2) * p.tiles_x + (int)(x >> p.ts_log2);
    if (!DT_IN_BOUNDS(j >= p.tile_e0 && j - p.tile_e0 < 512 && tile < p.tiles_per_plane, p.bounds)) return false;
    const int32_t s = p.tile_slot[(j - p.tile_e0) * p.tiles_per_plane + tile];
    if (s < 0) return false;
    if (!DT_IN_BOUNDS(s < p.tile_capacity, p.bounds)) return false;
    const uint32_t m = (1u << p.ts_log2) - 1u;
    const uint32_t k = ((y & m) << p.ts_log2) + (x & m);
    const float *t = p.tile_buf + (int64_t)s * p.slot_floats;
    f = ld_pixel_cached(t + k);
    if (PLANE_VAR) v = ld_pixel_cached(t + (1u << (2 * p.ts_log2)) + k);
    return true;
}

// One pixel of the extended stack (any store: resident planes, interleaved (flux, var), or device-mapped
// host planes): fp32 values widened to fp64; v is the exposure's scalar in scalar-variance mode.
template <bool PLANE_VAR>
__device__ __forceinline__ void load_pixel_any(const GatherParams &p, int64_t j, int64_t a, double v_scalar, double &f,
                                               double &v)
{
    if (p.flux_ptrs) {
        float ff, vv = 0.f;
        if (p.tile_slot && load_pixel_tiled<PLANE_VAR>(p, j, (uint32_t)a, ff, vv)) {
            f = (double)ff;
            v = PLANE_VAR ? (double)vv : v_scalar;
            return;
        }
        f = (double)ld_pixel_cached(p.flux_ptrs[j] + a);
        v = PLANE_VAR ? (double)ld_pixel_cached(p.var_ptrs[j] + a) : v_scalar;
    } else if (PLANE_VAR && p.fv) {
        const float2 t2 = ld_pixel2_cached(p.fv + (j * p.plane + a));
        f = (double)t2.x;
        v = (double)t2.y;
    } else {
        f = (double)ld_pixel_cached(p.flux + (j * p.plane + a));
        v = PLANE_VAR ? (double)ld_pixel_cached(p.var + (j * p.plane + a)) : v_scalar;
    }
}

// EXT: the extended stack of SURVEY 8(f) NEXT-1 / NEXT-3 (dtrack.h dt_set_patch, dt_set_outlier_clip): per
// intersection the k x k patch around the nearest pixel, row by row, s_i += (w f) / v, wt_i += (w w) / v over
// the valid pixels inside the image ("a patch of pixels is pulled"), the intersection dropped
// when s_i > clip sqrt(wt_i), else S += s_i, Wt += wt_i.  Every operation is an explicit
// round-to-nearest intrinsic (no contraction), in the order the definition states: bit-identical sums.
template <bool PLANE_VAR, bool EXT>
__global__ void __launch_bounds__(kSparseThreads) k_gather_sparse(const GatherParams p)
{
    if (gather_regime(p) != p.walk_form) return;
    const int lane = threadIdx.x & 31;
    const int64_t orbit = (int64_t)blockIdx.x * kSparseThreads + threadIdx.x;
    if (orbit >= p.n_pad) return;   // n_pad is a multiple of 32: whole warps leave together
    const int64_t tile = orbit >> 5;
    const int64_t n_tiles = p.n_pad >> 5;
    const unsigned lt = (1u << lane) - 1u;
    const bool cached = p.ld_cached != 0;

    double S = 0.0, Wt = 0.0;
    int32_t cnt = 0;
    bool touched = false;

    for (int g = 0; g < p.n_groups; ++g) {
        uint32_t bits = p.mask[(int64_t)g * p.n_pad + orbit];
        const uint32_t blk0 = (uint32_t)p.base[(int64_t)g * n_tiles + tile];   // independent of the mask: in flight with it
        if (!__any_sync(0xffffffffu, bits != 0u)) continue;
        // ---- column masks (lane jj holds exposure jj's: bit L = orbit L hits it) and the entry index of
        // each column: a 32 x 32 bit-matrix transpose across the warp in five butterfly steps (r2 profile:
        // the 32-ballot form was 65 % of all instructions this kernel executed) ----
        const uint32_t col = transpose32(bits, lane);
        const int c = __popc(col);
        int incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += v;
        }
        const uint32_t pre = blk0 + (uint32_t)(incl - c);
        const int64_t j0 = (int64_t)p.first_exposure + (int64_t)g * kGroup;
        if (bits && !touched) {
            // carry across exposure units: start from the partial sums of the earlier units so the
            // additions happen in exactly ascending-exposure order
            S = p.S[orbit];
            Wt = p.Wt[orbit];
            cnt = p.cnt[orbit];
            touched = true;
        }
        if constexpr (EXT) {
            const int h = p.patch >> 1;
            while (__any_sync(0xffffffffu, bits != 0u)) {
                const bool have = bits != 0u;
                const int jj = have ? __ffs(bits) - 1 : 0;
                bits &= bits - 1u;
                const uint32_t cj = __shfl_sync(0xffffffffu, col, jj);
                const uint32_t pj = __shfl_sync(0xffffffffu, pre, jj);
                if (have && DT_IN_BOUNDS((int64_t)(pj + __popc(cj & lt)) < p.offsets_cap, p.bounds)) {
                    const uint32_t off = p.offsets[pj + __popc(cj & lt)] & kOffsetMask;
                    if (!DT_IN_BOUNDS((int64_t)off < p.plane && j0 + jj < p.n_exp_store, p.bounds)) continue;
                    const int iy = (int)(off / (uint32_t)p.width), ix = (int)(off - (uint32_t)iy * (uint32_t)p.width);
                    const int64_t j = j0 + jj;
                    const double v_scalar = PLANE_VAR ? 0.0 : p.exp_all[j].var;
                    double si = 0.0, wti = 0.0;
                    int used = 0;
                    for (int dy = -h; dy <= h; ++dy) {
                        const int yy = iy + dy;
                        if (yy < 0 || yy >= p.height) continue;
                        for (int dx = -h; dx <= h; ++dx) {
                            const int xx = ix + dx;
                            if (xx < 0 || xx >= p.width) continue;
                            double f, v;
                            load_pixel_any<PLANE_VAR>(p, j, (int64_t)yy * p.width + xx, v_scalar, f, v);
                            if (isfinite(f) && isfinite(v) && v > 0.0) {
                                const double w = p.patch_w ? p.patch_w[(dy + h) * p.patch + (dx + h)] : 1.0;
                                si = __dadd_rn(si, __ddiv_rn(__dmul_rn(w, f), v));
                                wti = __dadd_rn(wti, __ddiv_rn(__dmul_rn(w, w), v));
                                used += 1;
                            }
                        }
                    }
                    if (used > 0 && !(si > __dmul_rn(p.clip, __dsqrt_rn(wti)))) {
                        S = __dadd_rn(S, si);
                        Wt = __dadd_rn(Wt, wti);
                        cnt += 1;
                    }
                }
            }
            continue;
        }
        while (__any_sync(0xffffffffu, bits != 0u)) {
            int jj[4];
            uint32_t idx[4], off[4];
            float f[4], vv[4];
            bool have[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                have[q] = bits != 0u;
                jj[q] = have[q] ? __ffs(bits) - 1 : 0;
                bits &= bits - 1u;                       // 0 stays 0
                const uint32_t cj = __shfl_sync(0xffffffffu, col, jj[q]);
                const uint32_t pj = __shfl_sync(0xffffffffu, pre, jj[q]);
                idx[q] = pj + __popc(cj & lt);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                have[q] = have[q] && DT_IN_BOUNDS((int64_t)idx[q] < p.offsets_cap, p.bounds);
                off[q] = have[q] ? (p.offsets[idx[q]] & kOffsetMask) : 0u;
                have[q] = have[q] && DT_IN_BOUNDS((int64_t)off[q] < p.plane && j0 + jj[q] < p.n_exp_store, p.bounds);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                f[q] = 0.f;
                vv[q] = 1.f;
                if (have[q]) {
                    if (p.flux_ptrs) {
                        // streaming mode: from the tile cache when the pixel's tile is resident, else
                        // zero-copy: straight from page-locked host memory over PCIe
                        if (!(p.tile_slot && load_pixel_tiled<PLANE_VAR>(p, j0 + jj[q], off[q], f[q], vv[q]))) {
                            f[q] = ld_pixel_cached(p.flux_ptrs[j0 + jj[q]] + off[q]);
                            if (PLANE_VAR) vv[q] = ld_pixel_cached(p.var_ptrs[j0 + jj[q]] + off[q]);
                        }
                    } else if (PLANE_VAR && p.fv) {
                        // a miss fetches 64 B of DRAM in the one-launch walk (no other hit of the line will find it in
                        // the L2: half the bytes at the same access rate) and the whole 128-B line in the slab form, where
                        // the line's other hits come by while it is resident: fewer DRAM accesses, which is what bounds
                        const float2 *a2 = p.fv + ((j0 + jj[q]) * p.plane + off[q]);
                        const float2 t2 = (p.walk_form == 2) ? ld_pixel2_cached(a2) : ld_pixel2_64(a2);
                        f[q] = t2.x;
                        vv[q] = t2.y;
                    } else {
                        const int64_t a = (j0 + jj[q]) * p.plane + off[q];
                        if (cached) {
                            f[q] = ld_pixel_64(p.flux + a);
                            if (PLANE_VAR) vv[q] = ld_pixel_64(p.var + a);
                        } else {
                            f[q] = ld_pixel_stream(p.flux + a);
                            if (PLANE_VAR) vv[q] = ld_pixel_stream(p.var + a);
                        }
                    }
                }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (have[q]) {
                    double v, w;
                    if (PLANE_VAR) {
                        v = (double)vv[q];
                        w = 1.0 / v;
                    } else {
                        const ExpRec &x = p.exp_all[j0 + jj[q]];
                        v = x.var;
                        w = x.inv_var;
                    }
                    // f / v from RN(1/v) with two FMA corrections (dt_gather.cuh): the bits of the IEEE division
                    if (v > 1e-150 && v < 1e150 && fabsf(f[q]) <= 3.402823466e38f) {
                        S += div_by_reciprocal((double)f[q], v, w);
                        Wt += w;
                        cnt += 1;
                    } else {
                        stack_one((double)f[q], v, w, S, Wt, cnt);
                    }
                }
            }
        }
    }
    if (touched && orbit < p.n_orbits) {
        p.S[orbit] = S;
        p.Wt[orbit] = Wt;
        p.cnt[orbit] = cnt;
    }
}

cudaError_t launch_gather(const GatherParams &p_in, int device, cudaStream_t stream)
{
    if (p_in.n_orbits <= 0 || p_in.n_groups <= 0) return cudaSuccess;
    GatherParams p = p_in;
    if (p.window < 1) p.window = 1;
    // schedules: 0 orbit-major walk (k_gather_sparse; the only one that reads device-mapped HOST planes),
    // 1 dense lock-step, -1: both are enqueued and each returns at once unless the unit's hit density, read on
    // the device, is in its regime
    // the extended stack (patch, weights, outlier clip) exists in the orbit-major walk only
    const bool ext = p.patch > 1 || p.patch_w != nullptr || isfinite(p.clip);
    if (p.patch < 1) p.patch = 1;
    if (p.flux_ptrs || ext) p.lockstep_mode = 0;
    if (p.lockstep_mode != 1) {
        const unsigned blocks = (unsigned)((p.n_pad + kSparseThreads - 1) / kSparseThreads);
        const bool plane_var = p.var || p.var_ptrs || p.fv;
        if (ext && plane_var)
            k_gather_sparse<true, true><<<blocks, kSparseThreads, 0, stream>>>(p);
        else if (ext)
            k_gather_sparse<false, true><<<blocks, kSparseThreads, 0, stream>>>(p);
        else if (plane_var)
            k_gather_sparse<true, false><<<blocks, kSparseThreads, 0, stream>>>(p);
        else
            k_gather_sparse<false, false><<<blocks, kSparseThreads, 0, stream>>>(p);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (p.lockstep_mode != 0 && !p.skip_dense) return launch_gather_dense(p, device, stream);
    return cudaSuccess;
}

cudaError_t init_device_kernels(int device, int *sm_count)
{
    cudaError_t e = cudaDeviceGetAttribute(sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    if ((e = init_propagate_kernels()) != cudaSuccess) return e;
    return init_gather_dense_kernels();
}

// ---- interleaved store ------------------------------------------------------------------------------------
__global__ void k_interleave(const float *__restrict__ flux, const float *__restrict__ var, float2 *__restrict__ dst,
                             int64_t n)
{
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x)
        dst[k] = make_float2(flux[k], var[k]);
}

cudaError_t launch_interleave(const float *flux, const float *var, float2 *dst, int64_t n, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    const unsigned blocks = (unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16);
    k_interleave<<<blocks, 256, 0, stream>>>(flux, var, dst, n);
    return cudaGetLastError();
}

// ---- finalisation ---------------------------------------------------------------------------------------
__global__ void k_finalize(const double *__restrict__ elements, const double *__restrict__ t0_orbit, int64_t n,
                           const double *__restrict__ S,
                           const double *__restrict__ Wt, const int32_t *__restrict__ cnt,
                           double *__restrict__ snr, int32_t *__restrict__ hits,
                           unsigned long long *invalid_counter)
{
    const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool bad = false;
    if (o < n) {
        const double *el = elements + o * 6;
        bool fin = true;
#pragma unroll
        for (int k = 0; k < 6; ++k) fin = fin && isfinite(el[k]);
        if (t0_orbit) fin = fin && isfinite(t0_orbit[o]);
        const bool valid = fin && el[0] > 0.0 && el[1] >= 0.0 && el[1] < 1.0;
        bad = !valid;
        const int32_t c = cnt[o];
        snr[o] = valid ? ((c > 0) ? S[o] / sqrt(Wt[o]) : 0.0) : nan("");
        hits[o] = valid ? c : -1;
    }
    const unsigned nb = __popc(__ballot_sync(0xffffffffu, bad));
    if ((threadIdx.x & 31) == 0 && nb && invalid_counter) atomicAdd(invalid_counter, (unsigned long long)nb);
}

cudaError_t launch_finalize(const double *elements, const double *t0_orbit, int64_t n, const double *S,
                            const double *Wt, const int32_t *cnt, double *snr, int32_t *hits,
                            unsigned long long *invalid_counter, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    k_finalize<<<blocks, 256, 0, stream>>>(elements, t0_orbit, n, S, Wt, cnt, snr, hits, invalid_counter);
    return cudaGetLastError();
}

}  // namespace dt
