// dt_k1.cuh -- everything kernel 1 (+2) is compiled from besides dt_orbit.cuh / dt_tma.cuh: the per-exposure record,
// its parameter block, the hit-entry format, the bounds-check macro.  Kept apart from dt_common.cuh so that the hash
// that ties bench.py's FP64 instruction counts to the kernel-1 sources (k1_counts.py) changes only when kernel 1 can.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

// Debug build (-DDT_BOUNDS_CHECK; `python -m paper_2503_08854_b200._build --bounds` -> libdtrack_bounds.so):
// every data-dependent index of kernels 1 - 3 and of the tile kernels is checked on the device; a violation is
// counted (counters[7]) and skipped, and the call that ran the kernel fails with DT_ERR_CUDA.  compute-sanitizer
// is closed on the GPU pool this was developed on (profiles/r2_memcheck.md); this is its stand-in.
#ifdef DT_BOUNDS_CHECK
#define DT_IN_BOUNDS(cond, ctr) ((cond) ? true : ((ctr) ? (atomicAdd((ctr), 1ull), false) : false))
#else
#define DT_IN_BOUNDS(cond, ctr) true
#endif

namespace dt {

// ---- per-exposure constant record ("a few hundred bytes of data for each image") ---
// 128 B = one TMA bulk-copy granule multiple; 32 records (one exposure group) = 4 KB in shared
// memory.  Observer and tangent basis are already rotated to the EQUATORIAL frame and the in-plane
// basis is divided by the pixel scale, so kernel 1 needs three dot products and one reciprocal.
struct __align__(16) ExpRec {
    double t;              // exposure mid-time, days
    double Rx, Ry, Rz;     // observer, heliocentric equatorial, AU
    double ex, ey, ez;     // east unit vector / pixel_scale   (x = cx + (q.e)/(q.t))
    double nx, ny, nz;     // north unit vector / pixel_scale  (y = cy + (q.n)/(q.t))
    double tx, ty, tz;     // unit vector to the tangent point (D = q.t)
    double var;            // scalar variance (mode 0); NaN in plane mode
    double inv_var;        // 1.0 / var (IEEE division on the host)
    double pad;
};
static_assert(sizeof(ExpRec) == 128, "ExpRec must be 128 bytes");

constexpr int kGroup = 32;          // exposures per group: one hit bit per exposure in a 32-bit mask
#ifndef DT_K1_TILE
#define DT_K1_TILE 128
#endif
constexpr int kTileOrbits = DT_K1_TILE;   // orbits per CTA of kernel 1 (one orbit per thread); 128 x 4 CTAs/SM
                                          // measured 7 % (MBA) to 11 % (NEO) faster than 256 x 2 and 192 x 3
constexpr int kWarpsPerCta = kTileOrbits / 32;

// ---- kernel 1 (+2): propagate, project, cull, compact ------------------------------------------
struct GatePolicy;
struct PropagateParams {
    const double *elements;     // [n][6], 16-B aligned; device memory or device-mapped pinned host memory
    double *elements_copy;      // NULL, or device [n][6]: the kernel leaves a copy of what it read
    int64_t n_orbits;           // orbits in this unit
    int64_t n_pad;              // n_orbits rounded up to 32 (mask row pitch)
    const ExpRec *exp;          // records of the unit's first exposure
    int32_t n_exp;              // exposures in this unit
    int32_t groups_per_split;   // exposure groups handled by one blockIdx.y
    double t0, gm, inv_c;       // inv_c = 0 disables light-time
    const double *t0_orbit;     // NULL, or device [n]: per-orbit epoch of M0 (dt_stack_epochs; replaces t0)
    double cos_eps, sin_eps;
    double cx, cy, W, H;        // (W-1)/2, (H-1)/2, width, height as fp64
    int32_t width;
    double tan_fov;             // tan of the footprint half-diagonal, for the conservative pre-cull
    // outputs of the cull + compaction stage (hit list format: dtrack.h dt_gather_hits)
    uint32_t *mask;             // [n_groups][n_pad]
    unsigned long long *base;   // [n_groups][n_pad/32]
    uint32_t *offsets;          // [capacity]
    int64_t offsets_cap;        // entries `offsets` can hold (bounds-check build)
    unsigned long long *counters;  // [0] unit hit allocator, [1] refined pairs, [2] cold solves, [3] hits, [4] sub-step solves, [6] gated pairs, [7] bounds violations
    const GatePolicy *policy;   // NULL, or: the kernel returns at once unless policy->select says its variant runs
    float4 *group_bounds;       // NULL, or device [3 x exposure groups of the launch]: written by launch_propagate
                                // (k_group_bounds) for the gate variant's group-level test (dt_orbit.cuh group_is_far)
    // dense debug outputs (dt_project), NULL on the timed path
    double *radec, *xy;         // [n][n_exp][2]
    int32_t *pix;               // [n][n_exp][2]
};

enum { kModeWarm = 1, kModePrecull = 2, kModeDense = 4, kModeGate = 8 };   // kModeGate: with kModeWarm | kModePrecull only

// Device-side choice between the kernel-1 variants with and without the group ephemeris gate (dt_orbit.cuh): both are
// enqueued for every unit and the one `select[0]` does not name returns at once, so the choice needs no host
// synchronisation.  k_gate_policy (dt_propagate.cu) sets it after every unit from what that unit did.
struct GatePolicy {
    int32_t select;                 // 1: the next unit runs the gate variant
    int32_t cooldown;               // units left before a gate that proved useless is tried again
    unsigned long long refined0, gated0;   // counters[1], counters[6] at the end of the previous unit
};
// max_unit_hits: NULL, or a word in device-mapped page-locked HOST memory that holds the largest hit count of any unit
// the context has processed: a hint the host reads, without synchronising, to decide which forms of kernel 3 are
// worth enqueueing at all (dt_api.cu launch_gather_unit); never a result.
cudaError_t launch_gate_policy(GatePolicy *policy, const unsigned long long *counters, int64_t unit_pairs,
                               unsigned long long *max_unit_hits, cudaStream_t stream);

cudaError_t launch_propagate(const PropagateParams &p, int mode, cudaStream_t stream);

// A hit entry is (exposure within its group) << kOffsetBits | (iy * W + ix): an entry names its exposure, so
// a block of the list can be processed as one flat coalesced list.  W * H <= 2^27 (dt_create checks).
constexpr int kOffsetBits = 27;
constexpr uint32_t kOffsetMask = (1u << kOffsetBits) - 1u;

}  // namespace dt
