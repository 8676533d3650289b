// dt_gather.cu -- kernel 3: gather + stack, and the SNR finalisation.
//
// Hot-path steps 8-9 of DESIGN.md (Algorithm 1 `FindLocalSignal` + the per-orbit combination,
// PAPER.md:171-172, 182 "jointly combining the signal from all intersections").  The paper pulls
// pixels on the CPU from mmap'd SSD files; here the images are in HBM.
//
// Mapping: the hit list is orbit-major (dtrack.h, dt_gather_hits).  One orbit per lane; a warp owns
// the same 32 orbits kernel 1's warp owned.  Per exposure group a lane reads its 32-bit hit mask
// (one coalesced 128-B row per warp), a warp scan of popcounts locates its run of pixel offsets,
// and it walks its own hits in ASCENDING exposure order accumulating S += f/v, Wt += 1/v in fp64
// REGISTERS -- no atomics, no shared memory, and the same summation order as the definition, so S
// and Wt are bit-identical to a sequential evaluation.  All warps sweep the groups in the same
// order, which bins the image reads by exposure (L2 locality); loads are issued four hits at a time
// to keep several sectors in flight per lane.
#include "dt_common.cuh"

namespace dt {

constexpr int kGatherThreads = 256;

__device__ __forceinline__ float ld_stream(const float *p)
{
    // read-only path, no L1 allocation: a pixel is used once per hit; reuse, if any, is in L2
    float v;
    asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}

template <bool PLANE_VAR>
__global__ void __launch_bounds__(kGatherThreads) k_gather_stack(const GatherParams p)
{
    const int lane = threadIdx.x & 31;
    const int64_t orbit = (int64_t)blockIdx.x * kGatherThreads + threadIdx.x;
    if (orbit >= p.n_pad) return;   // n_pad is a multiple of 32: whole warps leave together
    const bool in_range = orbit < p.n_orbits;
    const int64_t tile = orbit >> 5;
    const int64_t n_tiles = p.n_pad >> 5;

    double S = 0.0, Wt = 0.0;
    int32_t cnt = 0;
    bool touched = false;

    for (int g = 0; g < p.n_groups; ++g) {
        uint32_t bits = p.mask[(int64_t)g * p.n_pad + orbit];
        const unsigned any = __ballot_sync(0xffffffffu, bits != 0u);
        if (!any) continue;
        const int c = __popc(bits);
        int incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += v;
        }
        const unsigned long long b0 = p.base[(int64_t)g * n_tiles + tile];
        const uint32_t *offs = p.offsets + b0 + (unsigned long long)(incl - c);
        const int64_t j0 = (int64_t)p.first_exposure + (int64_t)g * kGroup;
        if (bits && !touched) {
            // carry across exposure units: start from the partial sums of the earlier units so the
            // additions happen in exactly ascending-exposure order (bit-identical to the definition)
            S = p.S[orbit];
            Wt = p.Wt[orbit];
            cnt = p.cnt[orbit];
            touched = true;
        }

        int k = 0;
        while (bits) {
            // up to four hits in flight
            int jj[4];
            uint32_t off[4];
            float f[4], vv[4];
            int m = 0;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (bits) {
                    jj[q] = __ffs(bits) - 1;
                    bits &= bits - 1;
                    off[q] = offs[k + q];
                    m = q + 1;
                } else {
                    jj[q] = 0;
                    off[q] = 0;
                }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (q < m) {
                    const int64_t a = (j0 + jj[q]) * p.plane + off[q];
                    f[q] = ld_stream(p.flux + a);
                    if (PLANE_VAR) vv[q] = ld_stream(p.var + a);
                }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (q < m) {
                    const double fd = (double)f[q];
                    double v, w;
                    if (PLANE_VAR) {
                        v = (double)vv[q];
                        w = 1.0 / v;
                    } else {
                        const ExpRec &x = p.exp_all[j0 + jj[q]];
                        v = x.var;
                        w = x.inv_var;
                    }
                    if (isfinite(fd) && isfinite(v) && v > 0.0) {
                        S += fd / v;
                        Wt += w;
                        cnt += 1;
                    }
                }
            }
            k += m;
        }
    }
    if (in_range && touched) {
        p.S[orbit] = S;
        p.Wt[orbit] = Wt;
        p.cnt[orbit] = cnt;
    }
}

cudaError_t launch_gather(const GatherParams &p, cudaStream_t stream)
{
    if (p.n_orbits <= 0 || p.n_groups <= 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((p.n_pad + kGatherThreads - 1) / kGatherThreads);
    if (p.var)
        k_gather_stack<true><<<blocks, kGatherThreads, 0, stream>>>(p);
    else
        k_gather_stack<false><<<blocks, kGatherThreads, 0, stream>>>(p);
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
