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

// 32 x 32 bit-matrix transpose across a warp: lane L holds row L (bit j = element (L, j)); returns, in lane j,
// column j (bit L = element (L, j)).  Five butterfly steps: at distance d the two lanes of a pair swap the
// off-diagonal d x d blocks of their 2d x 2d tile.  All 32 lanes must call.
__device__ __forceinline__ uint32_t transpose32(uint32_t x, int lane)
{
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
        const uint32_t m = (d == 16) ? 0x0000ffffu : (d == 8) ? 0x00ff00ffu : (d == 4) ? 0x0f0f0f0fu
                         : (d == 2) ? 0x33333333u : 0x55555555u;
        const uint32_t y = __shfl_xor_sync(0xffffffffu, x, d);
        x = (lane & d) ? ((x & ~m) | ((y & ~m) >> d)) : ((x & m) | ((y & m) << d));
    }
    return x;
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

// Regime of a unit's hit list, decided on the device from kernel 1's hit counter (grid-uniform):
//   1 dense    at least one hit per 16 pixels of every plane the unit covers: most 128-B lines of a plane are
//              touched, so the one-exposure-at-a-time lock-step that keeps the plane L2-resident pays;
//   2 slabs    a long list (>= kSlabMinHits per unit; tno+focused: 6.7e7 hits on 1.85e7 lines): the orbit-major
//              walk, launched once per slab of two exposure groups -- the kernel boundaries keep all warps within 64
//              exposures of each other, so a line is fetched from DRAM once for most of its hits instead of once
//              per hit (measured 1.02 -> 0.65 ms per unit); the launches cost ~6 us each, which a short list
//              (small_mba+focused: 0.15 ms per unit) cannot pay;
//   0 sparse   everything else: the orbit-major walk in one launch.
__device__ __forceinline__ int gather_regime(const GatherParams &p)
{
    if (p.lockstep_mode == 1) return 1;
    if (p.lockstep_mode == 0 && p.slab_mode >= 0) return p.slab_mode;
    const unsigned long long n_hits = p.n_hits_dev ? *p.n_hits_dev : (unsigned long long)p.n_hits_host;
    const int ug = p.unit_groups > 0 ? p.unit_groups : p.n_groups;
    if (p.lockstep_mode < 0 && n_hits * 16ull >= (unsigned long long)ug * kGroup * (unsigned long long)p.plane) return 1;
    if (p.slab_mode >= 0) return p.slab_mode;
    return n_hits >= kSlabMinHits ? 2 : 0;
}
__device__ __forceinline__ bool gather_is_dense(const GatherParams &p) { return gather_regime(p) == 1; }

// ---- lock-step throttle primitives of the persistent schedules (no data travels through them) ----
__device__ __forceinline__ int ld_relaxed(const int *p)
{
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void prefetch_l2(const void *p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
__device__ __forceinline__ void red_add_relaxed(int *p, int v)
{
    asm volatile("red.relaxed.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// pixel loads of the orbit-major walk: a miss fetches 64 B from DRAM instead of the default 128 B (measured
// with ncu on B200: 127 B per random 4-B gather by default, 64 B with the hint; profiles/r2_probes.md)
__device__ __forceinline__ float ld_pixel_64(const float *p)
{
    float v;
    asm volatile("ld.global.nc.L2::64B.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 ld_pixel2_64(const float2 *p)
{
    float2 v;
    asm volatile("ld.global.nc.L2::64B.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

// shared memory the persistent schedules may ask for: (S, Wt, cnt) of kMaxTilesPerWarp tiles per warp
// + one arrival counter per exposure (or window) of a unit
constexpr size_t kPersistentSmemMax = (size_t)kMaxTilesPerWarp * kGatherThreads * 20 + (512 + 36) * sizeof(int);

cudaError_t persistent_geometry(int64_t n_pad, int32_t n_groups, int sm_count, int *grid, int *tiles_per_warp,
                                size_t *smem);
cudaError_t launch_gather_dense(const GatherParams &p, int device, cudaStream_t stream);
cudaError_t init_gather_dense_kernels();

}  // namespace dt
