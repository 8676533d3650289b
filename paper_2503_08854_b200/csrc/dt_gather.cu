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
#include <algorithm>

#include "dt_common.cuh"
#include "dt_gather.cuh"

namespace dt {

constexpr int kSparseThreads = 256;

template <bool PLANE_VAR>
__global__ void __launch_bounds__(kSparseThreads) k_gather_sparse(const GatherParams p)
{
    if (gather_is_dense(p)) return;
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
        if (!__any_sync(0xffffffffu, bits != 0u)) continue;
        // ---- column masks (lane jj holds exposure jj's) and the entry index of each column ----
        uint32_t col = 0;
#pragma unroll
        for (int jj = 0; jj < 32; ++jj) {
            const unsigned b = __ballot_sync(0xffffffffu, (bits >> jj) & 1u);
            if (lane == jj) col = b;
        }
        const int c = __popc(col);
        int incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += v;
        }
        const uint32_t pre = (uint32_t)p.base[(int64_t)g * n_tiles + tile] + (uint32_t)(incl - c);
        const int64_t j0 = (int64_t)p.first_exposure + (int64_t)g * kGroup;
        if (bits && !touched) {
            // carry across exposure units: start from the partial sums of the earlier units so the
            // additions happen in exactly ascending-exposure order
            S = p.S[orbit];
            Wt = p.Wt[orbit];
            cnt = p.cnt[orbit];
            touched = true;
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
            for (int q = 0; q < 4; ++q) off[q] = have[q] ? p.offsets[idx[q]] : 0u;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                f[q] = 0.f;
                vv[q] = 1.f;
                if (have[q]) {
                    if (p.flux_ptrs) {
                        // zero-copy: the pixel comes straight from page-locked host memory over PCIe
                        f[q] = ld_pixel_cached(p.flux_ptrs[j0 + jj[q]] + off[q]);
                        if (PLANE_VAR) vv[q] = ld_pixel_cached(p.var_ptrs[j0 + jj[q]] + off[q]);
                    } else if (PLANE_VAR && p.fv) {
                        const float2 t2 = ld_pixel2_cached(p.fv + ((j0 + jj[q]) * p.plane + off[q]));
                        f[q] = t2.x;
                        vv[q] = t2.y;
                    } else {
                        const int64_t a = (j0 + jj[q]) * p.plane + off[q];
                        if (cached) {
                            f[q] = ld_pixel_cached(p.flux + a);
                            if (PLANE_VAR) vv[q] = ld_pixel_cached(p.var + a);
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
                    stack_one((double)f[q], v, w, S, Wt, cnt);
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
    if (p.lockstep_mode != 1) {
        const unsigned blocks = (unsigned)((p.n_pad + kSparseThreads - 1) / kSparseThreads);
        if (p.var || p.var_ptrs || p.fv)
            k_gather_sparse<true><<<blocks, kSparseThreads, 0, stream>>>(p);
        else
            k_gather_sparse<false><<<blocks, kSparseThreads, 0, stream>>>(p);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (p.lockstep_mode != 0) return launch_gather_dense(p, device, stream);
    return cudaSuccess;
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
__global__ void k_finalize(const double *__restrict__ elements, int64_t n, const double *__restrict__ S,
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
        const bool valid = fin && el[0] > 0.0 && el[1] >= 0.0 && el[1] < 1.0;
        bad = !valid;
        const int32_t c = cnt[o];
        snr[o] = valid ? ((c > 0) ? S[o] / sqrt(Wt[o]) : 0.0) : nan("");
        hits[o] = valid ? c : -1;
    }
    const unsigned nb = __popc(__ballot_sync(0xffffffffu, bad));
    if ((threadIdx.x & 31) == 0 && nb && invalid_counter) atomicAdd(invalid_counter, (unsigned long long)nb);
}

cudaError_t launch_finalize(const double *elements, int64_t n, const double *S, const double *Wt,
                            const int32_t *cnt, double *snr, int32_t *hits,
                            unsigned long long *invalid_counter, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    k_finalize<<<blocks, 256, 0, stream>>>(elements, n, S, Wt, cnt, snr, hits, invalid_counter);
    return cudaGetLastError();
}

}  // namespace dt
