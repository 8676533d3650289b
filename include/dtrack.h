/*
 * dtrack.h -- C ABI of the B200-native non-linear digital-tracking hot path.
 *
 * What the library computes (BASELINE.json north_star; the
 * paper gives the skeleton only: Algorithm 1 PAPER.md:149-176 `SearchImages` ->
 * `FilterGPUIntersections` -> `FindLocalSignal` -> combine -> `FindSignificantResults`, and
 * PAPER.md:141-143, 202 "orbital parameters -> sky position at the image time -> location within
 * the pixel grid -> keep intersections inside image bounds -> pull pixels -> jointly combine"):
 *
 *   for every candidate orbit o = (a, e, i, Omega, omega, M0 at epoch t0) and every exposure j
 *     1. n = sqrt(GM/a^3), M = M0 + n (t_j - t0), solve E - e sin E = M            (fp64)
 *     2. r = a(cos E - e) P + a sqrt(1-e^2) sin E Q          (heliocentric ecliptic)
 *     3. ONE light-time iteration: tau = |r(t_j) - R_j| / c, r' = r(t_j - tau); observer stays at t_j
 *     4. d = r' - R_j, rotate ecliptic -> equatorial by the obliquity
 *     5. gnomonic (TAN) projection about the exposure's tangent point, +x east, +y north,
 *        x = (W-1)/2 + xi/s, y = (H-1)/2 + eta/s, nearest pixel ix = floor(x + 1/2)
 *     6. cull unless D > 0 and 0 <= x + 1/2 < W and 0 <= y + 1/2 < H
 *     7. gather f = flux_j[iy][ix] and v = var_j[iy][ix] (or the exposure's scalar variance);
 *        skip the hit unless f, v finite and v > 0
 *     8. per orbit, ascending exposure: S += f/v, Wt += 1/v, hits += 1;  SNR = S / sqrt(Wt), 0 if
 *        hits == 0
 *   dt_topk: the k largest SNR (ties: lower orbit index first) among orbits with hits >= min_hits.
 *
 * Every step runs in hand-written sm_100a CUDA kernels; there is NO CPU fallback: every compute
 * call returns DT_ERR_CUDA when no CUDA device is usable.  Units: AU, days, radians.
 *
 * Conventions
 *   - every call returns a status: 0 = DT_OK, negative = error; nothing throws or aborts across
 *     the ABI.  dt_last_error(ctx) returns a context-owned, NUL-terminated string that stays valid
 *     until the next call on that context (a static string when ctx == NULL).
 *   - pointers are tagged by a `mem_kind` argument: DT_MEM_HOST (pageable host), DT_MEM_PINNED
 *     (page-locked host) or DT_MEM_DEVICE (device memory of the context's device).
 *   - ownership: dt_create copies all metadata; the caller owns every input and output buffer.
 *     The one exception is documented at dt_load_image_batch (streaming mode retains the pointer).
 *   - one context per host thread; no global state; a context is bound to one CUDA device/stream.
 */
#ifndef DTRACK_H
#define DTRACK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dt_context dt_context; /* opaque */

enum {
    DT_OK = 0,
    DT_ERR_INVALID_ARG = -1,
    DT_ERR_OOM = -2,
    DT_ERR_CUDA = -3,
    DT_ERR_NOT_LOADED = -4,
    DT_ERR_STATE = -5,
    DT_ERR_TOO_LARGE = -6      /* a size beyond a fixed capacity (dt_threshold_noalloc)            */
};
enum { DT_MEM_HOST = 0, DT_MEM_PINNED = 1, DT_MEM_DEVICE = 2 };

/* dt_survey.flags */
enum {
    DT_FLAG_FORCE_STREAM = 1,   /* never keep images resident: always stream batches from host     */
    DT_FLAG_KEPLER_COLD = 2,    /* solve every pair from a cold start with libdevice sincos        */
                                /* (reference mode of kernel 1; default is the warm-started solve) */
    DT_FLAG_NO_PRECULL = 4,     /* do the light-time refinement + projection for every pair, even  */
                                /* when a conservative cone test already proves a miss             */
    DT_FLAG_PROJECT_PRECULL = 8, /* dt_project runs kernel 1 exactly as dt_stack does, pre-cull and */
                                /* cull-quality Kepler chain included: a pair the cone test rejects */
                                /* is reported as culled (NaN, (-1,-1)).  For parity tests of the   */
                                /* path the timed kernel takes; default dt_project refines all.    */
    DT_FLAG_NO_GROUP_GATE = 16  /* never use the group ephemeris gate (one Kepler solve per orbit   */
                                /* and group of 32 exposures + a second-order Taylor position with  */
                                /* a rigorous remainder bound decide which pairs reach the per-pair */
                                /* Kepler step; results are identical with and without it)          */
};

/*
 * Exposure metadata (Algorithm 1 `image_list` + the per-image header record of PAPER.md:202,
 * "a few hundred bytes of data for each image").  All arrays are HOST pointers, copied by
 * dt_create.  All exposures share width x height (true of all five BASELINE.json configs).
 */
typedef struct {
    uint32_t struct_size;      /* sizeof(dt_survey): ABI versioning, must match                   */
    int32_t n_exposures;       /* N >= 1                                                          */
    int32_t width, height;     /* pixels; 1 <= W, H and W*H <= 2^27                               */
    const double *t;           /* [N] exposure mid-times, days                                    */
    const double *obs_ecl;     /* [N][3] heliocentric ECLIPTIC observer position at t[j], AU      */
    const double *ra0;         /* [N] tangent point right ascension, rad                          */
    const double *dec0;        /* [N] tangent point declination, rad                              */
    double pixel_scale;        /* rad per pixel, > 0                                              */
    double gm;                 /* AU^3/day^2; NaN => 2.959122082855911e-4 (Gaussian k^2)          */
    double c;                  /* AU/day; NaN => 173.14463267424033; +inf => no light-time        */
    double obliquity;          /* rad; NaN => 0.40909262775014904 (23.439281 deg)                 */
    int32_t variance_mode;     /* 0: per-exposure scalar var_scalar[N]; 1: fp32 plane per exposure */
    const double *var_scalar;  /* [N], mode 0 (ignored in mode 1)                                 */
    int32_t device;            /* CUDA device ordinal                                             */
    void *stream;              /* cudaStream_t supplied by the caller (e.g. torch's current       */
                               /* stream); NULL = the legacy default stream                       */
    int64_t hbm_budget_bytes;  /* device bytes the image store may use; 0 => 75% of free memory   */
    uint32_t flags;            /* DT_FLAG_*                                                       */
} dt_survey;

/* Counters of the most recent dt_stack call (dt_get_stats). */
typedef struct {
    uint32_t struct_size;
    int64_t n_orbits, n_exposures;
    int64_t pairs;             /* n_orbits * n_exposures                                          */
    int64_t hits;              /* footprint hits written by the cull+compaction stage             */
    int64_t invalid_orbits;    /* orbits rejected (a <= 0, e outside [0,1), non-finite)           */
    int64_t refined_pairs;     /* pairs that went through light-time refinement + projection      */
    int64_t cold_solves;       /* Kepler solves started cold (libdevice sincos Newton)            */
    int64_t substep_solves;    /* Kepler solves advanced by several warm sub-steps                */
    int64_t h2d_image_bytes;   /* image bytes streamed host -> device inside the call             */
    int32_t streamed;          /* 1 when the image store did not fit and batches were streamed    */
    int32_t n_image_batches;   /* exposure ranges processed                                       */
    float ms_total;            /* whole call, CUDA events on the context stream                   */
    float ms_propagate;        /* kernel 1+2 (propagate, project, cull, compact), summed          */
    float ms_gather;           /* kernel 3 (gather + stack), summed                               */
    float ms_finalize;         /* SNR finalisation                                                */
    int32_t launches;          /* kernels launched by the call                                    */
    int32_t propagate_launches, gather_launches;
    int32_t image_zero_copy;   /* 1 when a streamed survey was gathered straight from the pinned host     */
                               /* planes (few hits) instead of being copied batch by batch               */
    int32_t image_tiles;       /* 1 when a streamed survey went through the tiled image cache: only the   */
                               /* 64 x 64-pixel tiles the hits fall on were copied (h2d_image_bytes)       */
    int64_t tiles_fetched;     /* tiles copied host -> device by the call                                 */
    int64_t gated_pairs;       /* pairs the group ephemeris gate removed before any per-pair Kepler step  */
} dt_stats;

/*
 * dt_create: build a context for a survey.  Computes and uploads the per-exposure constant records
 * (observer rotated to the equatorial frame, tangent-plane basis scaled by 1/pixel_scale, variance).
 * Errors: DT_ERR_INVALID_ARG (NULL / size mismatch / non-positive sizes / non-finite metadata),
 * DT_ERR_CUDA (no device, or a CUDA call failed), DT_ERR_OOM.
 */
int dt_create(const dt_survey *survey, dt_context **out);
int dt_destroy(dt_context *ctx);

/*
 * dt_load_image_batch: register the difference images of exposures [first, first+count)
 * (Algorithm 1 `LoadImages`).  flux (and var in variance_mode 1, else NULL) point to
 * count contiguous planes [count][H][W] of fp32 in the memory named by mem_kind.
 *   - if the whole survey fits hbm_budget_bytes (and DT_FLAG_FORCE_STREAM is not set) the planes
 *     are COPIED into the context's image store in HBM and the caller may free them on return;
 *   - otherwise (streaming mode; north_star subsystem 4) the library RETAINS the pointers: they
 *     must be DT_MEM_PINNED (else DT_ERR_INVALID_ARG) and stay valid until dt_destroy or until the
 *     same exposure range is loaded again.  dt_stack then runs the search first (it needs no image) and
 *     moves only what the hits need: when a probe of the hit density predicts
 *     that the gathers would move less than 5 % of the bytes the planes hold (a blind search) no image is
 *     copied and the hit pixels are read straight from the (device-mapped) page-locked planes; otherwise
 *     the 64 x 64-pixel TILES the hits fall on are copied into a device tile cache (tiles with few hits stay
 *     zero-copy).  Planes that are not device-mappable (or "stream_tiles" = 0) are streamed whole, in
 *     double-buffered batches.  Results are bit-identical in every case (dt_stats.image_zero_copy,
 *     image_tiles, tiles_fetched, h2d_image_bytes say what was done).
 * Ranges may be loaded in any order and re-loaded; overlapping a previously loaded range replaces it.
 */
int dt_load_image_batch(dt_context *ctx, int32_t first_exposure, int32_t count, const float *flux,
                        const float *var, int32_t mem_kind);

/*
 * dt_stack: the hot path (steps 1-8 above) for n orbits against all exposures.
 *   elements  [n][6] = a (AU), e, i, Omega, omega, M0 (rad), fp64, in memory `mem_kind`
 *   t0        epoch of M0, days (one per call)
 *   snr_out   [n] fp64, hits_out [n] int32 (either may be NULL): device memory when mem_kind is
 *             DT_MEM_DEVICE, else host memory (pageable or page-locked; page-locked is faster)
 * DT_MEM_PINNED elements (16-byte aligned) are not copied to the device first: kernel 1 reads each
 * tile of 128 orbits with one bulk copy straight from the page-locked buffer while earlier tiles
 * compute, so the buffer must stay valid (and unchanged) until the call returns.
 * Invalid orbits do not fail the call: they get hits = -1, snr = NaN.  Results are complete when
 * the call returns (the call synchronises the context stream).  The per-orbit results also stay
 * on the device for dt_topk.  Errors: DT_ERR_NOT_LOADED unless every exposure has images.
 */
int dt_stack(dt_context *ctx, const double *elements, int64_t n, double t0, int32_t mem_kind,
             double *snr_out, int32_t *hits_out);

/*
 * dt_stack_epochs: dt_stack with ONE EPOCH PER ORBIT ("each of these curves is parametrized by six orbital
 * elements and an orbital epoch"): t0 [n] fp64, in the same memory
 * kind as `elements`; M = M0[o] + n[o] (t_j - t0[o]).  A non-finite epoch makes the orbit invalid
 * (hits = -1, snr = NaN).  Everything else as dt_stack.
 */
int dt_stack_epochs(dt_context *ctx, const double *elements, const double *t0, int64_t n, int32_t mem_kind,
                    double *snr_out, int32_t *hits_out);

/*
 * dt_set_patch: gather a k x k PATCH of pixels per intersection instead of the nearest pixel ("for each
 * valid intersection returned, a patch of pixels is pulled from the associated image", PAPER.md:143;
 * SURVEY.md 8(f) NEXT-1).  k odd, 1 .. 15; weights: HOST [k*k] fp64, row-major (dy, then dx), e.g. the PSF
 * sampled on the pixel grid, copied by the call; NULL = all 1.  For every intersection (nearest pixel
 * (ix, iy) inside the footprint), over the patch pixels p inside the image with finite f_p, v_p > 0, row by
 * row:  s_i += (w_p f_p) / v_p,  wt_i += (w_p w_p) / v_p;  an intersection without any valid pixel is
 * skipped, otherwise (subject to dt_set_outlier_clip) S += s_i, Wt += wt_i, hits += 1 in ascending exposure
 * order; SNR = S / sqrt(Wt).  k = 1 with NULL weights (the default) is the single-pixel stack, bit for bit.
 * Applies to the following dt_stack / dt_stack_epochs / dt_gather_hits calls.
 */
int dt_set_patch(dt_context *ctx, int32_t k, const double *weights);

/*
 * dt_set_outlier_clip: per-intersection outlier rejection ("Intersections with anomalously high SNR value
 * compared to the expectation can be removed"): an intersection whose
 * own SNR s_i / sqrt(wt_i) exceeds `clip` (tested as s_i > clip * sqrt(wt_i); single pixel: f/v >
 * clip * sqrt(1/v)) is dropped before the sums and not counted.  One-sided; +inf (default) switches it
 * off; NaN is DT_ERR_INVALID_ARG.
 */
int dt_set_outlier_clip(dt_context *ctx, double clip);

/*
 * dt_threshold: threshold mode of `FindSignificantResults` (Algorithm 1; "detections above an
 * SNR of 5"): every orbit of the most recent dt_stack with finite SNR >= snr_min and
 * hits >= min_hits, in ascending orbit index.  *n_found = how many there are; the first
 * min(*n_found, max_out) are written to the HOST arrays index_out [max_out] int64 and snr_out [max_out]
 * fp64 (snr_out may be NULL).  Errors: DT_ERR_STATE without a dt_stack result; DT_ERR_INVALID_ARG for NaN
 * snr_min or max_out < 0.
 */
int dt_threshold(dt_context *ctx, double snr_min, int32_t min_hits, int64_t max_out, int64_t *index_out,
                 double *snr_out, int64_t *n_found);

/*
 * dt_threshold_noalloc: threshold mode (as dt_threshold: Algorithm 1 `FindSignificantResults`, PAPER.md:173,
 * 336) for callers that cannot allocate -- code under CUDA graph capture, tight serving loops.  No context:
 * it works on the CURRENT device, on `stream` (a cudaStream_t passed as a plain pointer; NULL = default
 * stream), over the caller's DEVICE arrays snr_dev [n] fp64 and hits_dev [n] int32 (e.g. dt_stack's
 * DT_MEM_DEVICE outputs), and writes DEVICE outputs: *n_found_dev = how many orbits have finite SNR >=
 * snr_min and hits >= min_hits; index_out_dev [max_out] int64 and snr_out_dev [max_out] fp64 (may be NULL)
 * get the first min(*n_found_dev, max_out) of them in ascending orbit index (entries beyond that are left
 * untouched).  The call only enqueues work: no cudaMalloc / cudaFree or allocating library routine, no host
 * copy, no synchronisation; results are valid once `stream` has reached the end of the call's work, and the
 * caller owns every array it passes.
 * Scratch: a static device array of 16.0 MiB built into the library (every GPU that loads the library holds
 * it until the process exits), sized for n <= DT_NOALLOC_MAX_ORBITS; larger n is DT_ERR_TOO_LARGE (nothing
 * is enqueued).  All calls on a device share that array: calls must not overlap on the GPU (same stream, or
 * ordered by events) -- overlapping calls race.  Errors: DT_ERR_INVALID_ARG (NULL arrays, negative sizes, NaN
 * snr_min), DT_ERR_TOO_LARGE, DT_ERR_CUDA; dt_last_error(NULL) describes the last one.
 */
#define DT_NOALLOC_MAX_ORBITS 1048576
int dt_threshold_noalloc(void *stream, const double *snr_dev, const int32_t *hits_dev, int64_t n, double snr_min,
                         int32_t min_hits, int64_t max_out, int64_t *index_out_dev, double *snr_out_dev,
                         int64_t *n_found_dev);

/*
 * Exposure-sharded search.  The paper partitions the IMAGES across ranks without
 * replication; every rank searches all orbits against its images and "the results of these computations are
 * extremely sparse", so only the valid ones travel, asynchronously, to the process that owns the orbit
 * (PAPER.md:141, 204-210).  Here a rank's context is created on its exposure slice; after dt_stack the per-orbit
 * sums S = sum f/v, Wt = sum 1/v and the hit counts of that slice stay on the device, and
 *   dt_partials_sparse    compacts, on the device, the orbits with hits > 0 into (index ascending, S, Wt, hits)
 *                         lists -- what a rank sends; *n_found = how many there are (the first
 *                         min(*n_found, max_out) are written; outputs live in `mem_kind` memory);
 *   dt_partials_reset     zeroes the sums of the context;
 *   dt_partials_add       adds one such list (indices distinct, in [0, n)) to the sums: S[i] += S_in, ...;
 *                         calling it for the lists of ranks 0, 1, 2, ... in that order fixes the summation order
 *                         (ascending exposure slice), so every rank computes the same bits;
 *   dt_partials_finalize  SNR = S / sqrt(Wt) from the current sums (orbits the last dt_stack marked invalid stay
 *                         invalid), written to snr_out / hits_out (either may be NULL) and kept for dt_topk /
 *                         dt_threshold.
 * The definition this reaches: S = sum over slices (in order) of the slice's sequential sum -- the plain stack up to
 * the rounding of re-associated fp64 sums (<< the 1e-9 bar).  The exchange itself (one variable-length all-gather)
 * is torch.distributed plumbing in the binding (paper_2503_08854_b200/sharded.py).  All need a prior dt_stack on the
 * context (DT_ERR_STATE otherwise); n is that call's orbit count.
 */
int dt_partials_sparse(dt_context *ctx, int64_t max_out, int64_t *index_out, double *S_out, double *Wt_out,
                       int32_t *hits_out, int32_t mem_kind, int64_t *n_found);
int dt_partials_reset(dt_context *ctx);
int dt_partials_add(dt_context *ctx, const int64_t *index, const double *S, const double *Wt, const int32_t *hits,
                    int64_t m, int32_t mem_kind);
int dt_partials_finalize(dt_context *ctx, double *snr_out, int32_t *hits_out, int32_t mem_kind);

/*
 * dt_topk: the k largest SNR of the most recent dt_stack, SNR descending, ties by orbit index
 * ascending, over orbits with hits >= min_hits and finite SNR (Algorithm 1 `FindSignificantResults`,
 * PAPER.md:173).  index_out [k] int64, snr_out [k] fp64 are HOST pointers; *n_found = min(k, count).
 * Errors: DT_ERR_STATE when no dt_stack result exists; DT_ERR_INVALID_ARG for k < 0.
 */
int dt_topk(dt_context *ctx, int32_t k, int32_t min_hits, int64_t *index_out, double *snr_out,
            int32_t *n_found);

/*
 * dt_project: parity/debug entry (not on the timed path): steps 1-6 for every pair, written densely.
 *   radec_out [n][N][2] (alpha in [0, 2pi), delta), xy_out [n][N][2] (x, y), pix_out [n][N][2]
 *   ((-1,-1) when culled).  HOST pointers; any may be NULL.  Uses the same kernel template as
 *   dt_stack's kernel 1 (Kepler mode selected by the context flags); every pair is refined unless
 *   DT_FLAG_PROJECT_PRECULL is set, in which case the conservative pre-cull of dt_stack is kept and
 *   the pairs it rejects come back as NaN / (-1,-1).
 */
int dt_project(dt_context *ctx, const double *elements, int64_t n, double t0, double *radec_out,
               double *xy_out, int32_t *pix_out);

/*
 * dt_gather_hits: kernel 3 on a caller-supplied hit list (micro-benchmark / test entry).
 * The hit list uses the library's internal format for ONE exposure range
 * [first_exposure, first_exposure + 32*n_groups): for group g and orbit o, bit b of
 * mask[g*n_pad + o] says orbit o hits exposure first_exposure + 32 g + b; the pixel offsets
 * of warp-tile w = o/32 in group g start at offsets[base[g*(n_pad/32) + w]] and are ordered
 * exposure-ascending, then orbit-ascending inside the tile (so the hits of one exposure are
 * contiguous); an entry is (b << 27) | (iy*W + ix): it carries its exposure b within the group.  n_pad = n rounded up to 32; n <= 2^20, n_groups <= 16, fewer than 2^32 hits.
 * n_hits = number of entries of `offsets` (the kernel picks its dense lock-step or its sparse
 * schedule from the hit density).  All pointers are DEVICE pointers.
 * Accumulates into S[n], Wt[n] (fp64) and cnt[n] (int32), which the caller zero-initialises.
 * Images must be resident (DT_ERR_STATE in streaming mode).
 */
int dt_gather_hits(dt_context *ctx, int64_t n, int32_t first_exposure, int32_t n_groups,
                   const uint32_t *mask, const uint64_t *base, const uint32_t *offsets,
                   int64_t n_hits, double *S, double *Wt, int32_t *cnt);

/*
 * dt_filter_intersections: kernel 1 (+2) alone -- Algorithm 1 `SearchImages` + `FilterGPUIntersections`
 * -- for ONE work unit: orbits [0, n), n <= 2^20, against exposures
 * [first_exposure, first_exposure + n_exposures), n_exposures <= 512.  Needs no images.  Exposes the
 * compacted hit list in the format dt_gather_hits takes: *mask, *base, *offsets are DEVICE pointers
 * owned by the context, valid until the next dt_stack / dt_filter_intersections / dt_destroy on it;
 * *n_hits entries of *offsets, *n_pad = n rounded up to 32, *n_groups = ceil(n_exposures / 32).
 * Used by bench.py to time kernel 3 alone on the hit lists the search really produces and to count
 * their unique 32-B sectors (the bytes_min of the gather roofline).  Synchronises the context stream.
 */
int dt_filter_intersections(dt_context *ctx, const double *elements, int64_t n, double t0, int32_t mem_kind,
                            int32_t first_exposure, int32_t n_exposures, const uint32_t **mask,
                            const uint64_t **base, const uint32_t **offsets, int64_t *n_hits, int64_t *n_pad,
                            int32_t *n_groups);

/*
 * dt_sky_order: the order dt_stack processes one unit of orbits in (option "sort_orbits"; csrc/dt_sort.cu): position i
 * of the sorted unit holds orbit perm_out[i].  elements [n][6] fp64 and t0_orbit [n] (or NULL: the scalar t0) are
 * DEVICE arrays, n <= 2^20 (one unit), perm_out [n] uint32 a DEVICE array.  The key of an orbit is the equal-area
 * sky cell (512 x 2048) of its geometric direction from the observer at the survey's middle exposure (orbits with a
 * perihelion inside 0.7 AU sort after all others); the sort is
 * stable, so the permutation is a pure function of the input.  A measurement / test entry: the kernel-1 and
 * kernel-3 entries (dt_filter_intersections, dt_gather_hits) work on the order they are given, and a caller that
 * wants what dt_stack runs passes them elements[perm].  Synchronises the context stream.
 */
int dt_sky_order(dt_context *ctx, const double *elements_dev, const double *t0_orbit_dev, int64_t n, double t0,
                 uint32_t *perm_out_dev);

/*
 * dt_set_option: tuning knobs of a context (none changes any result; defaults are the measured best).
 *   "sort_orbits"         1 (default): dt_stack processes every unit of orbits in the order of where they are on the
 *                         sky at the survey's middle exposure (a device-side sort; sums are returned in the
 *                         caller's order), so that the 32 orbits of a warp are alike whatever order they were
 *                         listed in; 0: in the caller's order.  Results agree to rounding of the pixel
 *                         coordinates (1e-9 px), not bit for bit: which Kepler series a warp takes is a warp vote
 *   "group_gate"          -1 (default): for every work unit the device picks the kernel-1 variant with or without
 *                         the group ephemeris gate from what the previous unit did (on where warps cull -- a
 *                         blind search -- and the gate really gates; off where most pairs are refined or the
 *                         remainder bounds are loose); 0 never, 1 always
 *   "gather_schedule"     -1 chosen on the device from the hit density (default), 0 orbit-major walk,
 *                         1 dense lock-step (one exposure at a time)
 *   "gather_window"       dense schedule: exposures the fastest CTA may be ahead (0 = from the L2 size)
 *   "gather_prefetch"     dense schedule: planes ahead of the L2 prefetch sweep (0 = off)
 *   "gather_l1"           dense schedule: 1 pixel loads allocate in L1, 0 they do not
 *   "stream_tiles"        streaming mode: -1 / 1 use the tiled image cache when the planes are device-mappable
 *                         (default), 0 stream whole planes in double-buffered batches; "tile_min_hits": hits of
 *                         one orbit unit on a tile from which the tile is fetched (0 = tile bytes / 1024)
 *   "stream_zero_copy"    streaming mode: -1 probe the hit density (default), 0 always copy batches, 1 always
 *                         gather from the pinned planes
 *   "zero_copy_elements"  1 kernel 1 reads DT_MEM_PINNED elements in place (default), 0 copies them first
 * Errors: DT_ERR_INVALID_ARG for an unknown name or a value out of range.
 */
int dt_set_option(dt_context *ctx, const char *name, int64_t value);

int dt_get_stats(const dt_context *ctx, dt_stats *out);
const char *dt_last_error(const dt_context *ctx);

/* Library build information: "dtrack-b200 <version> sm_100a". */
const char *dt_version(void);

/*
 * dt_fp64_peak: measures the device's FP64 FMA issue rate with a register-resident DFMA loop
 * (the "alu" roofline denominator of kernel 1; MEASURED_PEAKS.json has no FP64 figure).
 * Writes achieved TFLOP/s (2 flop per DFMA) to *tflops.  device: CUDA ordinal.
 */
int dt_fp64_peak(int32_t device, double *tflops);

/*
 * dt_probe_random_gather: what the device gives a gather-bound kernel -- independent 4-B loads at hashed
 * addresses of a buffer of buffer_bytes (rounded down to a power of two; >= 1 MiB), eight in flight per thread;
 * hint64 != 0: the loads carry .L2::64B (a miss fetches 64 B of DRAM instead of 128 B).  Writes gathers per
 * second.  Over a buffer far beyond the L2 (8 GiB): the random-DRAM-access rate, the second roofline denominator
 * of kernel 3 on sparse hit lists; over a buffer that stays L2-resident (16 MiB, one 2048^2 plane): the rate of
 * fully divergent L2-hit gathers through the L1 miss path, the denominator of the dense schedule (DESIGN.md
 * "Measurement").
 */
int dt_probe_random_gather(int32_t device, int64_t buffer_bytes, int32_t hint64, double *gathers_per_s);

#ifdef __cplusplus
}
#endif
#endif /* DTRACK_H */
