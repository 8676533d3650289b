// dt_gather.cuh -- device helpers shared by the two schedules of kernel 3 (dt_gather.cu,
// dt_gather_dense.cu): pixel loads, the per-hit stacking arithmetic (DESIGN.md steps 9-10) and the
// regime decision.
#pragma once

#include "dt_common.cuh"

namespace dt {

// read-only path, no L1 allocation: with sparse hits a pixel is used once; reuse, if any, is in L2
__device__ __forceinline__ float ld_pixel_stream(const float *p)
{
    float v;
    asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
// read-only path with L1 allocation: in the reuse regime (many orbits per pixel) the few lines an
// exposure's hits fall in are then served per SM instead of hammering one L2 slice
__device__ __forceinline__ float ld_pixel_cached(const float *p)
{
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}

// (flux, variance) of one pixel of the interleaved store
__device__ __forceinline__ float2 ld_pixel2_cached(const float2 *p)
{
    float2 v;
    asm volatile("ld.global.nc.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

// Steps 9-10 for one hit: skipped (not counted) unless f, v finite and v > 0; w = 1/v.
__device__ __forceinline__ void stack_one(double f, double v, double w, double &S, double &Wt, int32_t &cnt)
{
    if (isfinite(f) && isfinite(v) && v > 0.0) {
        S += f / v;
        Wt += w;
        cnt += 1;
    }
}

// f / v from the correctly rounded reciprocal w = RN(1/v) with FMA corrections (Markstein): q0 = f w is
// within 1.5 ulp of f/v, one correction makes it faithful, the second gives the correctly rounded
// quotient -- the same bits as the IEEE division of the definition, without the divide sequence.
// Valid for finite f and v well inside the normal range (the caller checks).
__device__ __forceinline__ double div_by_reciprocal(double f, double v, double w)
{
    const double q0 = f * w;
    const double q1 = fma(fma(-q0, v, f), w, q0);
    return fma(fma(-q1, v, f), w, q1);
}

// Dense when the unit has at least one hit per 16 pixels of every plane it covers (then most 128-B
// lines of a plane are touched and keeping the plane L2-resident pays); grid-uniform.
__device__ __forceinline__ bool gather_is_dense(const GatherParams &p)
{
    if (p.lockstep_mode >= 0) return p.lockstep_mode == 1;
    const unsigned long long n_hits = p.n_hits_dev ? *p.n_hits_dev : (unsigned long long)p.n_hits_host;
    return n_hits * 16ull >= (unsigned long long)p.n_groups * kGroup * (unsigned long long)p.plane;
}

cudaError_t launch_gather_dense(const GatherParams &p, int device, cudaStream_t stream);

}  // namespace dt
