// dt_gather_dense.cu -- kernel 3, dense schedule: ONE persistent wave sweeping the exposures in
// lock-step (hot-path steps 8-9; Algorithm 1 `FindLocalSignal` + combine).
//
//   * Every orbit of the unit is owned by one lane for the whole launch: warp w of the grid owns the
//     warp-tiles (32 orbits, same tiles as kernel 1's warps) w, w + NW, w + 2 NW, ... (at most
//     kMaxTilesPerWarp), and the per-orbit accumulators S, Wt (fp64) and cnt live in SHARED memory at
//     a lane-private address -- no atomics, additions in ascending exposure order.
//   * The hit list is exposure-major inside a (warp-tile, group) block: for exposure jj the hitting
//     lanes' pixel offsets are contiguous in lane order, so a lane finds its entry with one ballot +
//     popc and the warp reads the offsets with ONE coalesced load.
//   * All warps of the grid walk the exposures in the same ascending order and a sliding window keeps
//     them together: nobody starts exposure j before every CTA has finished exposure j - window
//     (per-CTA arrival counters in shared memory, one global counter per exposure polled with relaxed
//     loads through a per-CTA cache -- a throttle, no data is communicated through it).  The planes
//     being gathered from are then a few consecutive exposures that stay L2-resident while ALL
//     orbits of the unit read them: a plane is fetched from DRAM once per launch instead of once per
//     wave of CTAs (profiles/r1a_baseline.md: 62.7 GB of DRAM reads for 8.9 GB of algorithmic bytes).
//     The grid is launched cooperatively so that all CTAs are co-resident (the throttle needs it).
#include "dt_common.cuh"
#include "dt_gather.cuh"

namespace dt {


// Shared memory of one CTA: (S, Wt) [T][kGatherThreads] double2, cnt [T][kGatherThreads] int32
// (accumulators, lane-private), arrive [n_local] int, done_upto int (lock-step throttle).
template <bool PLANE_VAR>
__global__ void __launch_bounds__(kGatherThreads, kGatherCtasPerSm) k_gather_dense(const GatherParams p)
{
    if (!gather_is_dense(p)) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int T = p.tiles_per_warp;
    constexpr int n_warps = kGatherThreads / 32;
    double2 *sAcc = reinterpret_cast<double2 *>(smem_raw);          // (S, Wt)
    int32_t *sC = reinterpret_cast<int32_t *>(sAcc + (size_t)T * kGatherThreads);
    int *arrive = sC + (size_t)T * kGatherThreads;
    const int n_local = p.n_groups * kGroup;
    volatile int *done_upto = arrive + n_local;   // exposures [0, done_upto) are finished by every CTA

    const int lane = threadIdx.x & 31;
    const int64_t NW = (int64_t)gridDim.x * n_warps;
    const int64_t gw = (int64_t)blockIdx.x * n_warps + (threadIdx.x >> 5);
    const int64_t n_tiles = p.n_pad >> 5;
    const unsigned lt = (1u << lane) - 1u;
    const int n_ctas = (int)gridDim.x;
    const bool cached = p.ld_cached != 0;

    for (int k = threadIdx.x; k <= n_local; k += kGatherThreads) arrive[k] = 0;   // and done_upto
    __syncthreads();

    // tiles this warp owns: gw + t NW, t < T (bit t of `owned`); this lane's orbit in tile t
    uint32_t owned = 0, touched = 0;
    bool spread = false;      // this warp's hits of the last exposure spanned more than half the plane
#pragma unroll
    for (int t = 0; t < kMaxTilesPerWarp; ++t)
        if (t < T && gw + (int64_t)t * NW < n_tiles) owned |= 1u << t;
    auto orbit_of = [&](int t) -> int64_t { return (gw + (int64_t)t * NW) * 32 + lane; };

    for (int g = 0; g < p.n_groups; ++g) {
        uint32_t bits[kMaxTilesPerWarp];
        uint32_t cur[kMaxTilesPerWarp];     // next unread entry of the (tile, group) block (warp-uniform)
        uint32_t any_bits = 0;
#pragma unroll
        for (int t = 0; t < kMaxTilesPerWarp; ++t) {
            bits[t] = 0;
            cur[t] = 0;
            if ((owned >> t) & 1u) {
                const int64_t o = orbit_of(t);
                bits[t] = p.mask[(int64_t)g * p.n_pad + o];
                cur[t] = (uint32_t)p.base[(int64_t)g * n_tiles + (o >> 5)];
                if (bits[t] && !((touched >> t) & 1u)) {
                    // carry across exposure units: start from the partial sums of the earlier units
                    const int a = t * kGatherThreads + threadIdx.x;
                    sAcc[a] = make_double2(p.S[o], p.Wt[o]);
                    sC[a] = p.cnt[o];
                    touched |= 1u << t;
                }
            }
            any_bits |= bits[t];
        }
        uint32_t gm = __reduce_or_sync(0xffffffffu, any_bits);   // exposures this warp has hits in

        // exposures without a hit in this warp are finished as far as the throttle is concerned
        if (!((gm >> lane) & 1u)) {
            const int jl = g * kGroup + lane;
            const int old = atomicAdd(&arrive[jl], 1);
            if (old == n_warps - 1) red_add_relaxed(p.progress + jl * kProgressStride, 1);
        }

        const int64_t j0 = (int64_t)p.first_exposure + (int64_t)g * kGroup;
        bool check_spread = true;
        while (gm) {
            const int jj = __ffs(gm) - 1;
            gm &= gm - 1;
            const int jl = g * kGroup + jj;
            // ---- throttle: every CTA has finished exposure jl - window ----
            const int need = jl - p.window;
            if (need >= 0) {
                int d = *done_upto;
                while (d <= need) {
                    if (ld_relaxed(p.progress + d * kProgressStride) >= n_ctas) {
                        d += 1;
                        if (lane == 0) atomicMax((int *)done_upto, d);
                    } else {
                        __nanosleep(40);
                        d = max(d, *done_upto);
                    }
                }
            }
            // ---- L2 prefetch of the next plane, when this warp's hits are spread over the plane ----
            // About half of the gathers of a uniformly hit plane are first touches of their line: DRAM
            // latency, and DRAM accessed line by line in gather order.  If the warp's hits of the
            // previous exposure spanned more than half the plane, every thread prefetches its share
            // (<= one 128-B line per thread and exposure) of the plane `prefetch` exposures ahead, which
            // then enters L2 as a sequential stream.  Clustered hit lists do not trigger it (a
            // whole-plane prefetch would waste DRAM bandwidth there).
            if (spread && p.first_exposure + jl + p.prefetch < p.n_exp_store) {
                const int64_t n_lines = (p.plane * (PLANE_VAR && p.fv ? 8 : 4) + 127) >> 7;
                const char *base = PLANE_VAR && p.fv
                                       ? reinterpret_cast<const char *>(p.fv + (j0 + jj + p.prefetch) * p.plane)
                                       : reinterpret_cast<const char *>(p.flux + (j0 + jj + p.prefetch) * p.plane);
                for (int64_t l = (int64_t)blockIdx.x * kGatherThreads + threadIdx.x; l < n_lines;
                     l += (int64_t)gridDim.x * kGatherThreads)
                    prefetch_l2(base + l * 128);
            }
            // ---- locate this lane's entry in each tile's block, read offsets (coalesced) ----
            uint32_t off[kMaxTilesPerWarp];
            uint32_t mine = 0;
#pragma unroll
            for (int t = 0; t < kMaxTilesPerWarp; ++t) {
                const bool h = (bits[t] >> jj) & 1u;
                const unsigned hm = __ballot_sync(0xffffffffu, h);
                const bool hb = h && DT_IN_BOUNDS((int64_t)(cur[t] + __popc(hm & lt)) < p.offsets_cap, p.bounds);
                off[t] = hb ? (p.offsets[cur[t] + __popc(hm & lt)] & kOffsetMask) : 0u;
                cur[t] += __popc(hm);
                mine |= (hb && DT_IN_BOUNDS((int64_t)off[t] < p.plane, p.bounds)) ? (1u << t) : 0u;
            }
            // ---- is this warp's hit set spread over the plane?  (predictor for the prefetch above;
            // re-evaluated on the first exposure of every group only: the reuse regime is issue-bound) ----
            if (p.prefetch > 0 && check_spread) {
                check_spread = false;
                uint32_t omin = 0xffffffffu, omax = 0u;
#pragma unroll
                for (int t = 0; t < kMaxTilesPerWarp; ++t) {
                    if ((mine >> t) & 1u) {
                        omin = min(omin, off[t]);
                        omax = max(omax, off[t]);
                    }
                }
                omin = __reduce_min_sync(0xffffffffu, omin);
                omax = __reduce_max_sync(0xffffffffu, omax);
                spread = omax > omin && (int64_t)(omax - omin) * 2 > p.plane;
            }
            const float *fplane = p.flux + (j0 + jj) * p.plane;
            const float *vplane = PLANE_VAR ? p.var + (j0 + jj) * p.plane : nullptr;
            float f[kMaxTilesPerWarp], vv[kMaxTilesPerWarp];
#pragma unroll
            for (int t = 0; t < kMaxTilesPerWarp; ++t) {
                f[t] = 0.f;
                vv[t] = 1.f;
                if ((mine >> t) & 1u) {
                    if (PLANE_VAR && p.fv) {
                        const float2 t2 = ld_pixel2_cached(p.fv + ((j0 + jj) * p.plane + off[t]));
                        f[t] = t2.x;
                        vv[t] = t2.y;
                    } else if (cached) {
                        f[t] = ld_pixel_cached(fplane + off[t]);
                        if (PLANE_VAR) vv[t] = ld_pixel_cached(vplane + off[t]);
                    } else {
                        f[t] = ld_pixel_stream(fplane + off[t]);
                        if (PLANE_VAR) vv[t] = ld_pixel_stream(vplane + off[t]);
                    }
                }
            }
            double vs = 1.0, ws = 1.0;
            bool fast = false;
            if (!PLANE_VAR) {
                const ExpRec &x = p.exp_all[j0 + jj];
                vs = x.var;
                ws = x.inv_var;
                fast = vs > 1e-150 && vs < 1e150;     // uniform; else the IEEE division of stack_one
            }
#pragma unroll
            for (int t = 0; t < kMaxTilesPerWarp; ++t) {
                if ((mine >> t) & 1u) {
                    const double v = PLANE_VAR ? (double)vv[t] : vs;
                    const double w = PLANE_VAR ? 1.0 / v : ws;
                    const int a = t * kGatherThreads + threadIdx.x;
                    if (fast) {
                        if (fabsf(f[t]) <= 3.402823466e38f) {   // finite (NaN compares false)
                            double2 acc = sAcc[a];
                            acc.x += div_by_reciprocal((double)f[t], vs, ws);
                            acc.y += ws;
                            sAcc[a] = acc;
                            sC[a] += 1;
                        }
                    } else {
                        double2 acc = sAcc[a];
                        int32_t c = sC[a];
                        stack_one((double)f[t], v, w, acc.x, acc.y, c);
                        sAcc[a] = acc;
                        sC[a] = c;
                    }
                }
            }
            // ---- arrival: this warp is done with exposure jl ----
            if (lane == 0) {
                const int old = atomicAdd(&arrive[jl], 1);
                if (old == n_warps - 1) red_add_relaxed(p.progress + jl * kProgressStride, 1);
            }
        }
    }
#pragma unroll
    for (int t = 0; t < kMaxTilesPerWarp; ++t) {
        if (((touched >> t) & 1u) && orbit_of(t) < p.n_orbits) {
            const int64_t o = orbit_of(t);
            const int a = t * kGatherThreads + threadIdx.x;
            const double2 acc = sAcc[a];
            p.S[o] = acc.x;
            p.Wt[o] = acc.y;
            p.cnt[o] = sC[a];
        }
    }
}

// Grid geometry: all CTAs co-resident (cooperative launch), as many warps as there are warp-tiles
// up to the machine's capacity, tiles spread evenly.
cudaError_t persistent_geometry(int64_t n_pad, int32_t n_groups, int sm_count, int *grid, int *tiles_per_warp,
                                size_t *smem)
{
    if (sm_count <= 0) return cudaErrorInvalidValue;
    constexpr int n_warps = kGatherThreads / 32;
    const int64_t n_tiles = n_pad >> 5;
    const int max_ctas = sm_count * kGatherCtasPerSm;
    int64_t ctas = (n_tiles + n_warps - 1) / n_warps;
    if (ctas > max_ctas) ctas = max_ctas;
    if (ctas < 1) ctas = 1;
    const int64_t NW = ctas * n_warps;
    int64_t T = (n_tiles + NW - 1) / NW;
    if (T < 1) T = 1;
    if (T > kMaxTilesPerWarp) return cudaErrorInvalidValue;   // unit larger than the kernel supports
    *grid = (int)ctas;
    *tiles_per_warp = (int)T;
    *smem = (size_t)T * kGatherThreads * 20 + ((size_t)n_groups * kGroup + 4) * sizeof(int);
    return cudaSuccess;
}

cudaError_t launch_gather_dense(const GatherParams &p_in, int device, cudaStream_t stream)
{
    GatherParams p = p_in;
    int grid = 0, T = 0;
    size_t smem = 0;
    (void)device;
    cudaError_t e = persistent_geometry(p.n_pad, p.n_groups, p.sm_count, &grid, &T, &smem);
    if (e != cudaSuccess) return e;
    p.tiles_per_warp = T;
    e = cudaMemsetAsync(p.progress, 0, (size_t)p.n_groups * kGroup * kProgressStride * sizeof(int), stream);
    if (e != cudaSuccess) return e;
    const bool plane_var = p.var || p.fv;
    const void *fn = plane_var ? (const void *)k_gather_dense<true> : (const void *)k_gather_dense<false>;
    void *args[] = {(void *)&p};
    return cudaLaunchCooperativeKernel(fn, dim3((unsigned)grid), dim3(kGatherThreads), args, smem, stream);
}

// dynamic shared memory opt-in (the accumulators of a full unit need up to ~166 KB), for the CURRENT device
cudaError_t init_gather_dense_kernels()
{
    cudaError_t e = cudaFuncSetAttribute(k_gather_dense<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)kPersistentSmemMax);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_gather_dense<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kPersistentSmemMax);
}

}  // namespace dt
