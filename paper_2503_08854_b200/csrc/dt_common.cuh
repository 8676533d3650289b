// dt_common.cuh -- shared declarations of the dtrack-b200 CUDA library (product code; shares
// nothing with oracle/).  Data layout in HBM, kernel parameter blocks, launcher prototypes.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "dt_k1.cuh"

namespace dt {

// ---- kernel 3: gather + stack ---------------------------------------------------------------------
struct GatherParams {
    int64_t n_orbits, n_pad;
    int32_t first_exposure;     // absolute index of the unit's first exposure
    int32_t n_groups;
    const uint32_t *mask;
    const unsigned long long *base;
    const uint32_t *offsets;
    const float *flux;          // plane of ABSOLUTE exposure j at flux + j * plane
    const float *var;           // same indexing; NULL in scalar mode
    // resident plane-variance store: flux and variance INTERLEAVED per pixel, (flux, var) of absolute
    // exposure j, pixel off at fv[j * plane + off]: one 8-B gather per hit instead of two 4-B gathers
    // into different planes (gathers are bound by the access rate, not by bytes); flux / var NULL then
    const float2 *fv;
    // zero-copy mode (sparse schedule only): per-exposure plane pointers, absolute index, device-mapped
    // page-locked HOST memory; flux / var above are NULL then
    const float *const *flux_ptrs;
    const float *const *var_ptrs;
    const ExpRec *exp_all;      // all exposure records (scalar variance), absolute index
    int64_t plane;              // pixels per plane
    double *S, *Wt;             // [n] running sums (read-modify-write once per launch)
    int32_t *cnt;               // [n]
    int *progress;              // [n_groups * 32 * kProgressStride] per-exposure count of CTAs done with it
    int32_t window;             // lock-step window: exposure j starts after j - window is finished
    int32_t tiles_per_warp;     // filled in by launch_gather
    const unsigned long long *n_hits_dev;   // hits of the unit on the device (kernel 1's counter) or NULL
    int64_t n_hits_host;        // used when n_hits_dev is NULL
    int32_t lockstep_mode;      // -1: decide from the hit density; 0: sparse schedule; 1: dense schedule
    // the orbit-major walk comes in two forms: one launch over the unit's groups (regime 0), or one launch per slab
    // of a few groups with the sums carried through S / Wt / cnt (regime 2): all warps are then within one slab of
    // each other and a line several orbits gather from is still in the L2 when the next orbit comes by
    int32_t slab_mode;          // -1: decide from the hit count; 0: one launch; 2: slabs
    int32_t walk_form;          // which form THIS launch of the walk is (0 or 2): it returns at once in the other regime
    int32_t unit_groups;        // exposure groups of the whole unit (a slab launch has fewer in n_groups)
    int32_t skip_dense;         // launch_gather: do not enqueue the dense schedule (the unit's first launch did)
    int32_t ld_cached;          // dense schedule: pixel loads allocate in L1 (1) or not (0)
    int32_t prefetch;           // dense schedule: planes ahead of the front that are prefetched into L2 (0 = off)
    int32_t n_exp_store;        // exposures the store holds from absolute index 0 (bound of the prefetch)
    int32_t sm_count;           // SMs of the context's device (grid of the persistent schedules)
    // extended stack (dtrack.h dt_set_patch, dt_set_outlier_clip): k x k patch
    // around the nearest pixel with PSF weights, per-intersection outlier rejection.  patch == 1, patch_w ==
    // NULL and clip == +inf is the plain single-pixel stack; anything else runs the orbit-major walk's
    // extended instantiation.
    int32_t patch;              // k >= 1, odd
    const double *patch_w;      // device [k*k] row-major, or NULL (all 1)
    double clip;                // +inf: no rejection
    int32_t width, height;      // image size (patch bounds, tile lookup)
    // tiled image cache (dt_tiles.cu; streaming mode): slot of tile (exposure - tile_e0, tile) or -1; a pixel
    // without a slot is read from flux_ptrs / var_ptrs (zero-copy).  NULL: no cache.
    const int32_t *tile_slot;   // [<= 512 exposures][tiles_per_plane]
    const float *tile_buf;      // slot s at tile_buf + s * slot_floats: ts*ts flux values, then ts*ts variances (plane mode)
    int64_t slot_floats;
    int32_t ts_log2, tiles_x, tiles_per_plane;
    int32_t tile_e0;            // absolute exposure of row 0 of tile_slot
    int32_t tile_capacity;      // slots of tile_buf (bounds-check build)
    int64_t offsets_cap;        // entries `offsets` holds (bounds-check build)
    unsigned long long *bounds; // violation counter of the bounds-check build (NULL: not counted)
};

// ---- tiled image cache of the streaming mode (dt_tiles.cu) -------------------------------------------------------
struct TileParams {
    int64_t n_pad;              // hit list of the unit (format: dtrack.h dt_gather_hits)
    int32_t n_groups;
    const uint32_t *mask;
    const unsigned long long *base;
    const uint32_t *offsets;
    int32_t n_exp;              // exposures of the unit (rows of tile_count / tile_slot in use)
    int32_t first_exposure;     // absolute index of the unit's first exposure (row 0)
    int32_t width, height, ts_log2, tiles_x, tiles_per_plane;
    int32_t *tile_count;        // [n_exp][tiles_per_plane], zero on entry and on exit
    int32_t *tile_slot;         // [n_exp][tiles_per_plane], -1 = not resident
    unsigned int *alloc;        // [0] slots handed out in this exposure unit, [1] fetch queue length, [2] tiles fetched (statistics)
    int32_t capacity;           // slots of tile_buf
    int32_t min_hits;           // a tile is fetched once a unit has at least this many hits on it
    uint2 *fetch_list;          // [capacity]: (row * tiles_per_plane + tile, slot)
    const float *const *flux_ptrs;   // device-mapped page-locked host planes, absolute exposure index
    const float *const *var_ptrs;    // NULL in scalar-variance mode
    float *tile_buf;
    int64_t slot_floats;
    int64_t offsets_cap;        // bounds-check build
    unsigned long long *bounds;
};
cudaError_t launch_tiles(const TileParams &t, int sm_count, cudaStream_t stream);



constexpr unsigned long long kSlabMinHits = 25000000ull;   // hits per unit from which the slab form pays
constexpr int kSlabGroups = 2;          // exposure groups per launch of the slab form of the walk (dt_gather.cuh)
constexpr int kProgressStride = 32;     // one 128-B line per exposure counter (no false sharing of polls)
#ifndef DT_K3_THREADS
#define DT_K3_THREADS 1024
#endif
constexpr int kGatherThreads = DT_K3_THREADS;   // threads per CTA of the dense schedule (1024: 4 % faster on the
                                                // uniform list than 512 x 2, 256 x 4, 128 x 8: fewer arrivals)
constexpr int kGatherCtasPerSm = 1024 / kGatherThreads;   // 1024 resident threads (64 registers each) per SM
constexpr int kMaxTilesPerWarp = 8;     // 148 SMs x 32 warps x 8 tiles x 32 orbits >= 2^20 orbits

cudaError_t launch_gather(const GatherParams &p, int device, cudaStream_t stream);
// Per-device kernel attributes (dynamic shared memory opt-in of every kernel of the library); called by
// dt_create after cudaSetDevice, so that a context on a second device of the same process is set up too.
cudaError_t init_device_kernels(int device, int *sm_count);
cudaError_t init_propagate_kernels();
cudaError_t init_gather_kernels();
// dst[k] = (flux[k], var[k]), k < n: builds the interleaved store from two device planes
cudaError_t launch_interleave(const float *flux, const float *var, float2 *dst, int64_t n, cudaStream_t stream);

// SNR finalisation: snr = S / sqrt(Wt) (0 when no hit), NaN / -1 for invalid orbits.
cudaError_t launch_finalize(const double *elements, const double *t0_orbit, int64_t n, const double *S,
                            const double *Wt, const int32_t *cnt, double *snr, int32_t *hits,
                            unsigned long long *invalid_counter, cudaStream_t stream);

// ---- device top-k (dt_topk.cu) ----------------------------------------------------------------------
struct TopkWorkspace {
    unsigned long long *keys = nullptr;    // [n] order-preserving keys (0 = excluded)
    unsigned long long *cand_key = nullptr;  // [cap] selected candidates
    long long *cand_idx = nullptr;
    unsigned int *hist = nullptr;          // [256] + scratch
    unsigned long long *state = nullptr;   // prefix / remaining-k state
    unsigned int *block_counts = nullptr;
    int64_t n_cap = 0, cand_cap = 0, blocks_cap = 0;
};

// Selects the k best (snr descending, index ascending) valid entries; writes them sorted to the
// host arrays.  Returns the number found through *n_found.
cudaError_t topk_device(const double *snr, const int32_t *hits, int64_t n, int32_t k,
                        int32_t min_hits, TopkWorkspace &ws, int64_t *index_out_host,
                        double *snr_out_host, int32_t *n_found, cudaStream_t stream);
void topk_free(TopkWorkspace &ws);
// sparse per-orbit partial sums of an exposure shard (dtrack.h dt_partials_*)
cudaError_t partials_sparse_device(const double *S, const double *Wt, const int32_t *cnt, int64_t n, int64_t max_out,
                                   TopkWorkspace &ws, long long *idx_out_dev, double *S_out_dev, double *Wt_out_dev,
                                   int32_t *cnt_out_dev, int64_t *n_found, cudaStream_t stream);
cudaError_t partials_add_device(const long long *idx, int64_t m, int64_t n, const double *S_in, const double *Wt_in,
                                const int32_t *cnt_in, double *S, double *Wt, int32_t *cnt, int *bad_dev,
                                cudaStream_t stream);
cudaError_t refinalize_device(int64_t n, const double *S, const double *Wt, const int32_t *cnt, double *snr,
                              int32_t *hits, cudaStream_t stream);
// Threshold mode: every valid entry (finite snr >= snr_min, hits >= min_hits) in ascending index order;
// *n_found = how many there are, the first min(*n_found, max_out) are written to the host arrays.
cudaError_t threshold_device(const double *snr, const int32_t *hits, int64_t n, double snr_min,
                             int32_t min_hits, int64_t max_out, TopkWorkspace &ws, int64_t *index_out_host,
                             double *snr_out_host, int64_t *n_found, cudaStream_t stream);

// The same without any allocation, host copy or synchronisation: scratch in a file-scope device array of dt_topk.cu,
// inputs and outputs DEVICE arrays (dtrack.h dt_threshold_noalloc); n <= threshold_noalloc_max().
cudaError_t threshold_noalloc_device(const double *snr, const int32_t *hits, int64_t n, double snr_min,
                                     int32_t min_hits, int64_t max_out, long long *index_out_dev,
                                     double *snr_out_dev, long long *n_found_dev, cudaStream_t stream);
int64_t threshold_noalloc_max();

// Sky order (dt_sort.cu): the permutation that sorts a unit's orbits by where they are on the sky at the key
// exposure, the sorted copies kernels 1 and 3 work on, and the way back for the per-orbit sums.
size_t sky_sort_temp_bytes(int64_t n_max);
cudaError_t sky_sort_unit(const double *elements, const double *t0_orbit, int64_t n, double t0, const ExpRec *key_exp,
                          double gm, double cos_eps, double sin_eps, uint32_t *keys_in, uint32_t *keys_out,
                          uint32_t *index_in, void *temp, size_t temp_bytes, uint32_t *perm, double *elements_sorted,
                          double *t0_sorted, cudaStream_t stream);
cudaError_t sky_unsort_sums(const uint32_t *perm, int64_t n, int64_t unit, const double *S_s, const double *Wt_s,
                            const int32_t *cnt_s, double *S, double *Wt, int32_t *cnt, cudaStream_t stream);

// FP64 FMA issue-rate probe (dt_fp64_peak).
cudaError_t fp64_peak_device(double *tflops, cudaStream_t stream);
// Random 4-B gather rate over a buffer of buffer_bytes (dt_probe_random_gather).
cudaError_t random_gather_probe(int64_t buffer_bytes, int hint64, double *gathers_per_s, cudaStream_t stream);

}  // namespace dt
