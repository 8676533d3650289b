// dt_api.cu -- the C ABI (include/dtrack.h): context, image store and batch scheduler, dt_stack
// orchestration, dt_project, dt_topk, statistics.  Host code only launches kernels and moves
// bytes; every step of the hot path runs in the kernels of dt_propagate.cu / dt_gather.cu /
// dt_topk.cu.  There is no CPU fallback: without a usable CUDA device every call fails.
#include "../../include/dtrack.h"

#include <math.h>
#include <stdarg.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <string>
#include <vector>

#include "dt_common.cuh"

using namespace dt;

namespace {

constexpr int64_t kMaxUnitOrbits = 1 << 20;   // orbits per work unit (bounds the hit buffer)
constexpr int32_t kMaxUnitExposures = 512;    // exposures per work unit (16 groups)
constexpr int kMinCtas = 148 * 4;             // fill the machine before giving up exposure splits
constexpr int kTileLog2 = 6;                  // streaming tile cache: 64 x 64-pixel tiles (16 KB of fp32 per plane)

struct Timer {
    cudaEvent_t a = nullptr, b = nullptr;
};

}  // namespace

struct dt_context {
    int device = 0;
    cudaStream_t stream = nullptr, copy_stream = nullptr;
    bool own_stream = false;
    int32_t N = 0, W = 0, H = 0;
    int64_t plane = 0;
    int32_t var_mode = 0;
    uint32_t flags = 0;
    double pixel_scale = 0, gm = 0, c = 0, inv_c = 0, obliq = 0, cos_eps = 1, sin_eps = 0, tan_fov = 0;
    std::vector<ExpRec> h_exp;
    ExpRec *d_exp = nullptr;

    // image store
    bool streaming = false;
    int64_t budget = 0;
    float *d_flux = nullptr, *d_var = nullptr;          // resident: N planes each (scalar-variance mode: flux only)
    float2 *d_fv = nullptr;                             // resident, plane-variance mode: (flux, var) interleaved per pixel
    std::vector<uint8_t> loaded;                        // per exposure
    std::vector<const float *> h_flux, h_var;           // streaming: retained pinned pointers
    float *d_buf_flux[2] = {nullptr, nullptr}, *d_buf_var[2] = {nullptr, nullptr};
    int32_t batch_exp = 0;
    cudaEvent_t ev_ready[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
    bool ev_free_recorded[2] = {false, false};

    // orbit-side buffers
    double *d_el = nullptr;
    int64_t el_cap = 0;
    double *d_t0 = nullptr;                             // per-orbit epochs of dt_stack_epochs
    int64_t t0_cap = 0;
    // sky order (dt_sort.cu): sorted copies kernels 1 and 3 work on, the permutation, the sort's scratch
    int32_t sort_orbits = 1;                            // option "sort_orbits"
    double *d_els = nullptr, *d_t0s = nullptr, *d_Ss = nullptr, *d_Wts = nullptr;
    int32_t *d_cnts = nullptr;
    uint32_t *d_perm = nullptr, *d_skey = nullptr;      // d_skey: [3][unit] keys in / keys out / index in
    void *d_sort_tmp = nullptr;
    int64_t els_cap = 0, t0s_cap = 0, Ss_cap = 0, Wts_cap = 0, cnts_cap = 0, perm_cap = 0, skey_cap = 0;
    size_t sort_tmp_bytes = 0;
    // extended stack (dt_set_patch, dt_set_outlier_clip)
    int32_t patch = 1;
    double *d_patch_w = nullptr;                        // [patch * patch] or NULL (all 1)
    double clip = INFINITY;
    double *d_S = nullptr, *d_Wt = nullptr, *d_snr = nullptr;
    int32_t *d_cnt = nullptr, *d_hits = nullptr;
    int64_t acc_cap = 0, n_last = -1;
    uint32_t *d_mask = nullptr;
    unsigned long long *d_base = nullptr;
    uint32_t *d_offsets = nullptr;
    int64_t mask_cap = 0, base_cap = 0, off_cap = 0;
    unsigned long long *d_counters = nullptr;           // [8]
    GatePolicy *d_policy = nullptr;                     // kernel-1 variant of the next unit (device-side choice)
    unsigned long long *h_max_hits = nullptr, *d_max_hits = nullptr;   // largest unit hit count seen: mapped host word
    float4 *d_group_bounds = nullptr;                   // [3 x exposure groups]: the gate's group-level bounds of a launch
    int32_t group_gate = -1;                            // -1 chosen on the device, 0 never, 1 always
    int32_t gather_slab = -1;                           // walk in slabs: -1 chosen on the device, 0 never, k: always, k groups
    int *d_progress = nullptr;                          // kernel 3 lock-step counters, one per exposure of a unit
    int32_t gather_window = 1;                          // exposures the slowest and fastest CTA may be apart
    int32_t gather_lockstep = -1;                       // schedule: -1 decided on the device from the hit density
    int32_t gather_ld_cached = 1;
    int32_t gather_prefetch = 1;                        // planes ahead (dense schedule, resident store)
    int32_t sm_count = 0;                               // SMs of this context's device
    int32_t stream_zero_copy = -1;                      // -1 decide from a probe, 0 never, 1 always
    const float **d_flux_ptrs = nullptr, **d_var_ptrs = nullptr;   // [N] device-mapped pinned planes (zero-copy gather)
    // streaming mode, tiled image cache (dt_tiles.cu)
    int32_t stream_tiles = -1;                          // -1 / 1: use it when the planes are device-mappable, 0: never
    int32_t tile_min_hits = 0;                          // 0: default (a tile's bytes / 256)
    int32_t *tile_count = nullptr, *tile_slot = nullptr;
    unsigned int *tile_alloc = nullptr;
    uint2 *tile_fetch = nullptr;
    float *tile_buf = nullptr;
    int32_t tile_capacity = 0, tiles_x = 0, tiles_per_plane = 0;
    int64_t slot_floats = 0;
    bool zero_copy_elements = true;                     // false: copy pinned elements to the device first
    std::vector<cudaEvent_t> ev_pool;                   // timing events
    std::vector<cudaEvent_t> ev_elem;                   // per orbit unit: its elements have arrived on the device

    // scratch of the dt_partials_* calls (host-memory callers)
    long long *d_pidx = nullptr;
    double *d_pS = nullptr, *d_pW = nullptr;
    int32_t *d_pc = nullptr;
    int64_t p_cap = 0;
    int *d_bad = nullptr;
    TopkWorkspace topk;
    dt_stats stats;
    std::string err;
};

namespace {

const char *g_static_err = "dtrack: invalid context";

int fail(dt_context *ctx, int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf;
    return code;
}

#define CU(ctx, call)                                                                          \
    do {                                                                                       \
        cudaError_t e__ = (call);                                                              \
        if (e__ != cudaSuccess)                                                                \
            return fail(ctx, e__ == cudaErrorMemoryAllocation ? DT_ERR_OOM : DT_ERR_CUDA,      \
                        "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__,     \
                        __LINE__);                                                             \
    } while (0)

template <typename T>
cudaError_t grow(T *&ptr, int64_t &cap, int64_t need)
{
    if (ptr && need <= cap) return cudaSuccess;
    if (ptr) cudaFree(ptr);
    ptr = nullptr;
    cap = 0;
    if (need <= 0) need = 1;
    cudaError_t e = cudaMalloc((void **)&ptr, (size_t)need * sizeof(T));
    if (e == cudaSuccess) cap = need;
    return e;
}

void free_all(dt_context *c)
{
    cudaFree(c->d_exp);
    cudaFree(c->d_flux);
    cudaFree(c->d_var);
    cudaFree(c->d_fv);
    for (int s = 0; s < 2; ++s) {
        cudaFree(c->d_buf_flux[s]);
        cudaFree(c->d_buf_var[s]);
        if (c->ev_ready[s]) cudaEventDestroy(c->ev_ready[s]);
        if (c->ev_free[s]) cudaEventDestroy(c->ev_free[s]);
    }
    cudaFree(c->d_el);
    cudaFree(c->d_t0);
    cudaFree(c->d_pidx);
    cudaFree(c->d_pS);
    cudaFree(c->d_pW);
    cudaFree(c->d_pc);
    cudaFree(c->d_bad);
    cudaFree(c->d_patch_w);
    cudaFree(c->d_S);
    cudaFree(c->d_Wt);
    cudaFree(c->d_snr);
    cudaFree(c->d_cnt);
    cudaFree(c->d_hits);
    cudaFree(c->d_mask);
    cudaFree(c->d_base);
    cudaFree(c->d_offsets);
    cudaFree(c->d_counters);
    cudaFree(c->d_els); cudaFree(c->d_t0s); cudaFree(c->d_Ss); cudaFree(c->d_Wts); cudaFree(c->d_cnts);
    cudaFree(c->d_perm); cudaFree(c->d_skey); cudaFree(c->d_sort_tmp);
    cudaFree(c->d_policy);
    cudaFree(c->d_group_bounds);
    if (c->h_max_hits) cudaFreeHost(c->h_max_hits);
    cudaFree(c->d_progress);
    cudaFree(c->tile_count);
    cudaFree(c->tile_slot);
    cudaFree(c->tile_alloc);
    cudaFree(c->tile_fetch);
    cudaFree(c->tile_buf);
    cudaFree((void *)c->d_flux_ptrs);
    cudaFree((void *)c->d_var_ptrs);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    for (cudaEvent_t e : c->ev_elem) cudaEventDestroy(e);
    topk_free(c->topk);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
}

// Per-exposure constant record (hot-path step 2): observer rotated to the equatorial frame,
// tangent-plane basis (east, north) divided by the pixel scale, tangent unit vector.
ExpRec make_record(const dt_context *c, double t, const double *obs, double ra0, double dec0, double var)
{
    ExpRec r;
    memset(&r, 0, sizeof r);
    r.t = t;
    r.Rx = obs[0];
    r.Ry = obs[1] * c->cos_eps - obs[2] * c->sin_eps;
    r.Rz = obs[1] * c->sin_eps + obs[2] * c->cos_eps;
    const double sa = sin(ra0), ca = cos(ra0), sd = sin(dec0), cd = cos(dec0);
    const double is = 1.0 / c->pixel_scale;
    r.ex = -sa * is;
    r.ey = ca * is;
    r.ez = 0.0;
    r.nx = -sd * ca * is;
    r.ny = -sd * sa * is;
    r.nz = cd * is;
    r.tx = cd * ca;
    r.ty = cd * sa;
    r.tz = sd;
    r.var = var;
    r.inv_var = 1.0 / var;
    return r;
}

// Lock-step window of kernel 3: the planes of window + 1 consecutive exposures (flux, and variance
// in plane mode) should stay L2-resident while every orbit of the unit reads them.  Half of the L2
// is budgeted (data read by SMs of both dies may be held once per die).  DT_GATHER_WINDOW overrides.
int32_t pick_gather_window(const dt_context *c)
{
    int l2 = 0;
    if (cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, c->device) != cudaSuccess || l2 <= 0) l2 = 64 << 20;
    const int64_t per_exp = c->plane * 4 * (c->var_mode == 1 ? 2 : 1);
    int64_t w = ((int64_t)l2 / 2) / std::max<int64_t>(per_exp, 1) - 1;
    return (int32_t)std::max<int64_t>(1, std::min<int64_t>(w, 16));
}

int mem_kind_ok(int32_t k) { return k == DT_MEM_HOST || k == DT_MEM_PINNED || k == DT_MEM_DEVICE; }

// Streaming mode, whole-plane double buffering: two device slots of batch_exp exposures each.
int ensure_stream_slots(dt_context *c)
{
    {
        if (c->d_buf_flux[0]) return DT_OK;
        if (c->tile_buf) {                    // the tile cache and the plane slots share the image budget
            cudaFree(c->tile_buf);
            c->tile_buf = nullptr;
            c->tile_capacity = 0;
        }
        const int64_t per_exp = c->plane * 4 * (c->var_mode == 1 ? 2 : 1);
        int64_t b = c->budget / (2 * per_exp);
        if (b < 1) return fail(c, DT_ERR_OOM, "hbm_budget_bytes %lld cannot hold two exposures of %lld bytes",
                               (long long)c->budget, (long long)per_exp);
        b = std::min<int64_t>(b, kMaxUnitExposures);
        b = std::min<int64_t>(b, c->N);
        if (b >= kGroup) b -= b % kGroup;
        c->batch_exp = (int32_t)b;
        for (int s = 0; s < 2; ++s) {
            CU(c, cudaMalloc((void **)&c->d_buf_flux[s], (size_t)(b * c->plane) * 4));
            if (c->var_mode == 1) CU(c, cudaMalloc((void **)&c->d_buf_var[s], (size_t)(b * c->plane) * 4));
            CU(c, cudaEventCreateWithFlags(&c->ev_ready[s], cudaEventDisableTiming));
            CU(c, cudaEventCreateWithFlags(&c->ev_free[s], cudaEventDisableTiming));
        }
        return DT_OK;
    }
}

// Streaming mode, tiled image cache (dt_tiles.cu): count / slot tables for one exposure unit and as many tile
// slots as the image budget holds.
int ensure_tile_cache(dt_context *c)
{
    const int32_t ts = 1 << kTileLog2;
    c->tiles_x = (c->W + ts - 1) / ts;
    c->tiles_per_plane = c->tiles_x * ((c->H + ts - 1) / ts);
    c->slot_floats = (int64_t)ts * ts * (c->var_mode == 1 ? 2 : 1);
    if (c->tile_buf) return DT_OK;
    for (int s = 0; s < 2; ++s) {             // the plane slots and the tile cache share the image budget
        cudaFree(c->d_buf_flux[s]);
        cudaFree(c->d_buf_var[s]);
        c->d_buf_flux[s] = c->d_buf_var[s] = nullptr;
    }
    const size_t cells = (size_t)kMaxUnitExposures * (size_t)c->tiles_per_plane;
    if (!c->tile_count) {
        CU(c, cudaMalloc((void **)&c->tile_count, cells * sizeof(int32_t)));
        CU(c, cudaMemsetAsync(c->tile_count, 0, cells * sizeof(int32_t), c->stream));
        CU(c, cudaMalloc((void **)&c->tile_slot, cells * sizeof(int32_t)));
        CU(c, cudaMalloc((void **)&c->tile_alloc, 8 * sizeof(unsigned int)));
        CU(c, cudaMemsetAsync(c->tile_alloc, 0, 8 * sizeof(unsigned int), c->stream));
    }
    int64_t cap = c->budget / (c->slot_floats * 4);
    cap = std::min<int64_t>(cap, (int64_t)cells);            // every tile of the unit resident: nothing more to gain
    if (cap < 1) return fail(c, DT_ERR_OOM, "hbm_budget_bytes %lld cannot hold one image tile", (long long)c->budget);
    CU(c, cudaMalloc((void **)&c->tile_buf, (size_t)cap * (size_t)c->slot_floats * 4));
    cudaFree(c->tile_fetch);
    c->tile_fetch = nullptr;
    CU(c, cudaMalloc((void **)&c->tile_fetch, (size_t)cap * sizeof(uint2)));
    c->tile_capacity = (int32_t)std::min<int64_t>(cap, 0x7fffffff);
    return DT_OK;
}

int ensure_store(dt_context *c)
{
    if (c->streaming) return DT_OK;           // streaming buffers are created by the path dt_stack takes
    if (c->var_mode == 1) {
        if (!c->d_fv) CU(c, cudaMalloc((void **)&c->d_fv, (size_t)(c->N * c->plane) * 8));
    } else if (!c->d_flux) {
        CU(c, cudaMalloc((void **)&c->d_flux, (size_t)(c->N * c->plane) * 4));
    }
    return DT_OK;
}

}  // namespace

extern "C" {

#ifdef DT_BOUNDS_CHECK
const char *dt_version(void) { return "dtrack-b200 0.2 sm_100a +bounds"; }
#else
const char *dt_version(void) { return "dtrack-b200 0.2 sm_100a"; }
#endif

const char *dt_last_error(const dt_context *ctx) { return ctx ? ctx->err.c_str() : g_static_err; }

int dt_create(const dt_survey *s, dt_context **out)
{
    if (!out) return DT_ERR_INVALID_ARG;
    *out = nullptr;
    if (!s || s->struct_size != sizeof(dt_survey)) return DT_ERR_INVALID_ARG;
    if (s->n_exposures < 1 || s->width < 1 || s->height < 1 ||
        (int64_t)s->width * s->height > ((int64_t)1 << kOffsetBits))
        return DT_ERR_INVALID_ARG;
    if (!s->t || !s->obs_ecl || !s->ra0 || !s->dec0) return DT_ERR_INVALID_ARG;
    if (!(s->pixel_scale > 0.0) || !isfinite(s->pixel_scale)) return DT_ERR_INVALID_ARG;
    if (s->variance_mode != 0 && s->variance_mode != 1) return DT_ERR_INVALID_ARG;
    if (s->variance_mode == 0 && !s->var_scalar) return DT_ERR_INVALID_ARG;
    for (int32_t j = 0; j < s->n_exposures; ++j) {
        if (!isfinite(s->t[j]) || !isfinite(s->ra0[j]) || !isfinite(s->dec0[j]) ||
            !isfinite(s->obs_ecl[3 * j]) || !isfinite(s->obs_ecl[3 * j + 1]) ||
            !isfinite(s->obs_ecl[3 * j + 2]))
            return DT_ERR_INVALID_ARG;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || s->device < 0 || s->device >= ndev) {
        cudaGetLastError();
        return DT_ERR_CUDA;   // no CPU fallback
    }
    dt_context *c = new (std::nothrow) dt_context();
    if (!c) return DT_ERR_OOM;
    memset(&c->stats, 0, sizeof c->stats);
    c->stats.struct_size = sizeof(dt_stats);
    c->device = s->device;
    if (cudaSetDevice(c->device) != cudaSuccess) { delete c; return DT_ERR_CUDA; }
    c->N = s->n_exposures;
    c->W = s->width;
    c->H = s->height;
    c->plane = (int64_t)s->width * s->height;
    c->var_mode = s->variance_mode;
    c->flags = s->flags;
    c->pixel_scale = s->pixel_scale;
    c->gm = isnan(s->gm) ? 2.959122082855911025e-4 : s->gm;
    c->c = isnan(s->c) ? 173.14463267424033 : s->c;
    c->obliq = isnan(s->obliquity) ? 0.40909262775014904 : s->obliquity;
    if (!(c->gm > 0.0) || !(c->c > 0.0)) { delete c; return DT_ERR_INVALID_ARG; }
    c->inv_c = isinf(c->c) ? 0.0 : 1.0 / c->c;
    c->cos_eps = cos(c->obliq);
    c->sin_eps = sin(c->obliq);
    c->tan_fov = 0.5 * c->pixel_scale * sqrt((double)c->W * c->W + (double)c->H * c->H);

    c->stream = (cudaStream_t)s->stream;   // NULL = the legacy default stream
    int rc = DT_OK;
    do {
        if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { rc = DT_ERR_CUDA; break; }
        c->h_exp.resize(c->N);
        for (int32_t j = 0; j < c->N; ++j) {
            const double v = (c->var_mode == 0) ? s->var_scalar[j] : nan("");
            c->h_exp[j] = make_record(c, s->t[j], s->obs_ecl + 3 * j, s->ra0[j], s->dec0[j], v);
        }
        if (cudaMalloc((void **)&c->d_exp, sizeof(ExpRec) * (size_t)c->N) != cudaSuccess) { rc = DT_ERR_OOM; break; }
        if (cudaMemcpyAsync(c->d_exp, c->h_exp.data(), sizeof(ExpRec) * (size_t)c->N, cudaMemcpyHostToDevice,
                            c->stream) != cudaSuccess) { rc = DT_ERR_CUDA; break; }
        if (cudaMalloc((void **)&c->d_counters, 8 * sizeof(unsigned long long)) != cudaSuccess) { rc = DT_ERR_OOM; break; }
        if (cudaMalloc((void **)&c->d_policy, sizeof(GatePolicy)) != cudaSuccess) { rc = DT_ERR_OOM; break; }
        if (cudaMalloc((void **)&c->d_group_bounds, sizeof(float4) * 3 * (size_t)((s->n_exposures + kGroup - 1) / kGroup + 1)) != cudaSuccess) { rc = DT_ERR_OOM; break; }
        if (cudaHostAlloc((void **)&c->h_max_hits, sizeof(unsigned long long), cudaHostAllocMapped) == cudaSuccess) {
            *c->h_max_hits = 0;
            if (cudaHostGetDevicePointer((void **)&c->d_max_hits, c->h_max_hits, 0) != cudaSuccess) c->d_max_hits = nullptr;
        }
        cudaGetLastError();                                       // without the word: no hint, every form is enqueued
        {
            const GatePolicy first = {1, 0, 0ull, 0ull};          // a context starts with the gate on
            if (cudaMemcpy(c->d_policy, &first, sizeof first, cudaMemcpyHostToDevice) != cudaSuccess) { rc = DT_ERR_CUDA; break; }
        }
        if (cudaMalloc((void **)&c->d_progress, (size_t)(kMaxUnitExposures + kGroup) * kProgressStride * sizeof(int)) != cudaSuccess) { rc = DT_ERR_OOM; break; }
        c->gather_window = pick_gather_window(c);
        // kernel attributes are per DEVICE: set them for this context's device (no process-wide statics)
        if (init_device_kernels(c->device, &c->sm_count) != cudaSuccess) { rc = DT_ERR_CUDA; break; }
        if (cudaStreamSynchronize(c->stream) != cudaSuccess) { rc = DT_ERR_CUDA; break; }
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { rc = DT_ERR_CUDA; break; }
        c->budget = s->hbm_budget_bytes > 0 ? s->hbm_budget_bytes : (int64_t)(0.75 * (double)free_b);
        const int64_t need = (int64_t)c->N * c->plane * 4 * (c->var_mode == 1 ? 2 : 1);
        c->streaming = (c->flags & DT_FLAG_FORCE_STREAM) || need > c->budget;
        c->loaded.assign(c->N, 0);
        if (c->streaming) {
            c->h_flux.assign(c->N, nullptr);
            c->h_var.assign(c->N, nullptr);
        }
    } while (0);
    if (rc != DT_OK) {
        cudaGetLastError();
        free_all(c);
        delete c;
        return rc;
    }
    *out = c;
    return DT_OK;
}

int dt_destroy(dt_context *c)
{
    if (!c) return DT_ERR_INVALID_ARG;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    if (c->copy_stream) cudaStreamSynchronize(c->copy_stream);
    free_all(c);
    delete c;
    return DT_OK;
}

int dt_load_image_batch(dt_context *c, int32_t first, int32_t count, const float *flux, const float *var,
                        int32_t mem_kind)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (first < 0 || count < 1 || (int64_t)first + count > c->N || !flux || !mem_kind_ok(mem_kind))
        return fail(c, DT_ERR_INVALID_ARG, "dt_load_image_batch: bad range or pointer");
    if (c->var_mode == 1 && !var) return fail(c, DT_ERR_INVALID_ARG, "variance_mode 1 needs a variance plane");
    CU(c, cudaSetDevice(c->device));
    if (c->streaming) {
        if (mem_kind != DT_MEM_PINNED)
            return fail(c, DT_ERR_INVALID_ARG,
                        "survey exceeds hbm_budget_bytes: streaming mode needs DT_MEM_PINNED images");
        for (int32_t j = 0; j < count; ++j) {
            c->h_flux[first + j] = flux + (int64_t)j * c->plane;
            c->h_var[first + j] = (c->var_mode == 1) ? var + (int64_t)j * c->plane : nullptr;
            c->loaded[first + j] = 1;
        }
        return DT_OK;
    }
    int rc = ensure_store(c);
    if (rc != DT_OK) return rc;
    if (c->var_mode == 1) {
        // plane-variance mode: the store interleaves (flux, var) per pixel.  Device sources are read in
        // place; host sources go through a staging buffer a few planes at a time.
        float2 *dst = c->d_fv + (int64_t)first * c->plane;
        if (mem_kind == DT_MEM_DEVICE) {
            CU(c, launch_interleave(flux, var, dst, (int64_t)count * c->plane, c->stream));
        } else {
            const int32_t chunk = std::min<int32_t>(count, 4);
            float *stage = nullptr;
            CU(c, cudaMalloc((void **)&stage, (size_t)chunk * (size_t)c->plane * 8));
            for (int32_t j = 0; j < count; j += chunk) {
                const int32_t m = std::min<int32_t>(chunk, count - j);
                const size_t b = (size_t)m * (size_t)c->plane * 4;
                cudaError_t e = cudaMemcpyAsync(stage, flux + (int64_t)j * c->plane, b, cudaMemcpyHostToDevice, c->stream);
                if (e == cudaSuccess)
                    e = cudaMemcpyAsync(stage + (int64_t)chunk * c->plane, var + (int64_t)j * c->plane, b,
                                        cudaMemcpyHostToDevice, c->stream);
                if (e == cudaSuccess)
                    e = launch_interleave(stage, stage + (int64_t)chunk * c->plane, dst + (int64_t)j * c->plane,
                                          (int64_t)m * c->plane, c->stream);
                if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
                if (e != cudaSuccess) {
                    cudaFree(stage);
                    return fail(c, DT_ERR_CUDA, "dt_load_image_batch: %s", cudaGetErrorString(e));
                }
            }
            cudaFree(stage);
        }
    } else {
        const size_t bytes = (size_t)count * (size_t)c->plane * 4;
        CU(c, cudaMemcpyAsync(c->d_flux + (int64_t)first * c->plane, flux, bytes, cudaMemcpyDefault, c->stream));
    }
    CU(c, cudaStreamSynchronize(c->stream));
    for (int32_t j = 0; j < count; ++j) c->loaded[first + j] = 1;
    return DT_OK;
}

static int propagate_mode(const dt_context *c)
{
    int mode = 0;
    if (!(c->flags & DT_FLAG_KEPLER_COLD)) mode |= kModeWarm;
    if (!(c->flags & DT_FLAG_NO_PRECULL)) mode |= kModePrecull;
    return mode;
}

// the call's counters restart from zero, and with them the policy's snapshots of two of them (its choice is kept)
static cudaError_t reset_counters(dt_context *c)
{
    cudaError_t e = cudaMemsetAsync(c->d_counters, 0, 8 * sizeof(unsigned long long), c->stream);
    if (e != cudaSuccess) return e;
    return cudaMemsetAsync(&c->d_policy->refined0, 0, 2 * sizeof(unsigned long long), c->stream);
}

// Kernel 1 of one unit.  The group ephemeris gate (dt_orbit.cuh) exists for the default mode only (warm chain +
// pre-cull); unless an option or a flag fixes it, BOTH variants are enqueued -- the one the device-side policy does
// not name returns at once -- and the policy is updated from what the unit did: no host synchronisation.
static cudaError_t launch_k1_unit(dt_context *c, PropagateParams &p, int mode, int32_t *launches)
{
    const bool can_gate = mode == (kModeWarm | kModePrecull);
    const int gate = (!can_gate || (c->flags & DT_FLAG_NO_GROUP_GATE)) ? 0 : c->group_gate;
    p.policy = nullptr;
    cudaError_t e;
    if (gate >= 0) {
        *launches += 2;
        e = launch_propagate(p, gate ? (mode | kModeGate) : mode, c->stream);
    } else {
        p.policy = c->d_policy;
        e = launch_propagate(p, mode | kModeGate, c->stream);
        if (e == cudaSuccess) e = launch_propagate(p, mode, c->stream);
        *launches += 3;
    }
    // one thread: the next unit's variant, and the largest unit hit count seen (the host's hint for kernel 3)
    if (e == cudaSuccess)
        e = launch_gate_policy(c->d_policy, c->d_counters, p.n_orbits * (int64_t)p.n_exp, c->d_max_hits, c->stream);
    return e;
}

// Kernel 3 of one unit: the dense schedule, the orbit-major walk in one launch, and the walk in slabs of exposure
// groups (dt_gather.cuh gather_regime).  Unless options fix the choice all are enqueued and every kernel that is not
// of the unit's regime -- read on the device from kernel 1's hit counter -- returns at once.
static cudaError_t launch_gather_unit(const dt_context *c, const GatherParams &g_in, int32_t *launches)
{
    GatherParams g = g_in;
    g.unit_groups = g.n_groups;
    const bool ext = g.patch > 1 || g.patch_w != nullptr || isfinite(g.clip);
    if (g.flux_ptrs || ext) g.lockstep_mode = 0;                       // as launch_gather: walk only
    int32_t slab_opt = c->gather_slab;                                 // -1 auto, 0 never, k > 0: always, k groups
    if (g.flux_ptrs || g.lockstep_mode == 1) slab_opt = 0;             // pixels over PCIe / dense forced: no slabs
    // the slab launches cost a few microseconds each even when they return at once: they are enqueued only once the
    // context has produced a unit with 80 % of the hits the slab regime takes (a hint read without synchronising:
    // a stale or missing value only changes which of two equivalent forms runs)
    if (slab_opt < 0 && c->h_max_hits && g.n_hits_dev &&
        *(volatile unsigned long long *)c->h_max_hits < kSlabMinHits / 5 * 4)
        slab_opt = 0;
    if (slab_opt < 0 && !g.n_hits_dev && (unsigned long long)g.n_hits_host < kSlabMinHits) slab_opt = 0;   // known here
    const int32_t slab = slab_opt > 0 ? slab_opt : kSlabGroups;
    if (slab_opt == 0 || slab >= g.n_groups) {
        g.slab_mode = 0;
        g.walk_form = 0;
        *launches += (g.lockstep_mode < 0) ? 2 : 1;
        return launch_gather(g, c->device, c->stream);
    }
    g.slab_mode = slab_opt > 0 ? 2 : -1;
    if (slab_opt < 0 || g.lockstep_mode < 0) {                         // the one-launch walk (and the dense schedule)
        g.walk_form = 0;
        cudaError_t e = launch_gather(g, c->device, c->stream);
        if (e != cudaSuccess) return e;
        *launches += (g.lockstep_mode < 0) ? 2 : 1;
    }
    g.walk_form = 2;
    g.skip_dense = 1;
    for (int32_t g0 = 0; g0 < g.unit_groups; g0 += slab) {
        GatherParams s = g;
        s.n_groups = std::min<int32_t>(slab, g.unit_groups - g0);
        s.mask = g.mask + (int64_t)g0 * g.n_pad;
        s.base = g.base + (int64_t)g0 * (g.n_pad >> 5);
        s.first_exposure = g.first_exposure + g0 * kGroup;
        cudaError_t e = launch_gather(s, c->device, c->stream);
        if (e != cudaSuccess) return e;
        *launches += 1;
    }
    return cudaSuccess;
}

static void fill_gather_ext(const dt_context *c, GatherParams &g)
{
    g.tile_capacity = c->tile_capacity;
    g.offsets_cap = g.offsets == c->d_offsets ? c->off_cap : (int64_t)1 << 40;   // dt_gather_hits: the caller's list
    g.bounds = c->d_counters + 7;
    g.patch = c->patch;
    g.patch_w = c->d_patch_w;
    g.clip = c->clip;
    g.width = c->W;
    g.height = c->H;
}

static void fill_common(const dt_context *c, PropagateParams &p, double t0)
{
    memset(&p, 0, sizeof p);
    p.t0 = t0;
    p.gm = c->gm;
    p.inv_c = c->inv_c;
    p.cos_eps = c->cos_eps;
    p.sin_eps = c->sin_eps;
    p.cx = 0.5 * ((double)c->W - 1.0);
    p.cy = 0.5 * ((double)c->H - 1.0);
    p.W = (double)c->W;
    p.H = (double)c->H;
    p.width = c->W;
    p.tan_fov = c->tan_fov;
    p.offsets_cap = c->off_cap;
    p.group_bounds = c->d_group_bounds;
}

static int32_t pick_groups_per_split(int64_t n_orbits, int32_t n_exp)
{
    const int64_t tiles = (n_orbits + kTileOrbits - 1) / kTileOrbits;
    const int32_t n_groups = (n_exp + kGroup - 1) / kGroup;
    if (tiles >= kMinCtas) return n_groups;
    int64_t splits = (kMinCtas + tiles - 1) / tiles;
    splits = std::min<int64_t>(splits, n_groups);
    return (int32_t)((n_groups + splits - 1) / splits);
}

}  // extern "C"

// dt_stack and dt_stack_epochs: t0_orbit == NULL means the scalar epoch t0
static int stack_impl(dt_context *c, const double *elements, const double *t0_orbit, int64_t n, double t0,
                      int32_t mem_kind, double *snr_out, int32_t *hits_out)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (n < 0 || (n > 0 && !elements) || !mem_kind_ok(mem_kind) || !isfinite(t0))
        return fail(c, DT_ERR_INVALID_ARG, "dt_stack: bad arguments");
    for (int32_t j = 0; j < c->N; ++j)
        if (!c->loaded[j]) return fail(c, DT_ERR_NOT_LOADED, "exposure %d has no image", j);
    CU(c, cudaSetDevice(c->device));
    int rc = ensure_store(c);
    if (rc != DT_OK) return rc;

    dt_stats &st = c->stats;
    memset(&st, 0, sizeof st);
    st.struct_size = sizeof(dt_stats);
    st.n_orbits = n;
    st.n_exposures = c->N;
    st.pairs = n * (int64_t)c->N;
    st.streamed = c->streaming ? 1 : 0;
    c->n_last = -1;
    if (n == 0) { c->n_last = 0; return DT_OK; }

    // ---- buffers ----
    // an exposure unit is at most 512 exposures; only the whole-plane streaming path uses smaller ones (its
    // double-buffered batches), decided below
    const int32_t unit_exp_max = std::min<int32_t>(c->N, kMaxUnitExposures);
    int32_t unit_exp = unit_exp_max;
    const int64_t unit_orb = std::min<int64_t>((n + 31) / 32 * 32, kMaxUnitOrbits);
    const int32_t unit_groups = (unit_exp_max + kGroup - 1) / kGroup;
    // Elements: kernel 1 stages each tile with one bulk copy, from device memory or straight from
    // page-locked host memory (first pass over the orbits; it leaves a device copy for later passes
    // and for the finalisation).  Pageable or misaligned inputs are copied to the device first.
    const double *d_el = elements;           // what later passes and k_finalize read
    const double *first_src = elements;      // what the first pass of kernel 1 reads
    double *copy_out = nullptr;
    bool elements_by_unit = false;           // the elements arrive unit by unit on the copy stream (ev_elem)
    const bool aligned16 = (reinterpret_cast<uintptr_t>(elements) & 15u) == 0;
    if (mem_kind != DT_MEM_DEVICE || !aligned16) {
        CU(c, grow(c->d_el, c->el_cap, n * 6));
        d_el = c->d_el;
        void *mapped = nullptr;
        if (mem_kind == DT_MEM_PINNED && aligned16 && c->zero_copy_elements && !c->sort_orbits &&
            cudaHostGetDevicePointer(&mapped, const_cast<double *>(elements), 0) == cudaSuccess && mapped &&
            (reinterpret_cast<uintptr_t>(mapped) & 15u) == 0) {
            first_src = static_cast<const double *>(mapped);
            copy_out = c->d_el;
        } else if (c->sort_orbits && mem_kind != DT_MEM_DEVICE) {
            // sky order needs a unit's elements on the device before its kernel 1: one copy per orbit unit on the
            // copy stream, all enqueued now, so that unit u + 1 crosses PCIe while unit u is being worked on
            cudaGetLastError();
            first_src = c->d_el;
            const int64_t units = (n + unit_orb - 1) / unit_orb;
            while ((int64_t)c->ev_elem.size() < units) {
                cudaEvent_t e;
                CU(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
                c->ev_elem.push_back(e);
            }
            for (int64_t u = 0; u < units; ++u) {
                const int64_t o0 = u * unit_orb, no = std::min<int64_t>(unit_orb, n - o0);
                CU(c, cudaMemcpyAsync(c->d_el + o0 * 6, elements + o0 * 6, (size_t)no * 48, cudaMemcpyHostToDevice,
                                      c->copy_stream));
                CU(c, cudaEventRecord(c->ev_elem[u], c->copy_stream));
            }
            elements_by_unit = true;
        } else {
            cudaGetLastError();
            CU(c, cudaMemcpyAsync(c->d_el, elements, (size_t)n * 48, cudaMemcpyDefault, c->stream));
            first_src = c->d_el;
        }
    }
    // per-orbit epochs: on the device before kernel 1 (8 B per orbit)
    const double *d_t0 = nullptr;
    if (t0_orbit) {
        if (mem_kind == DT_MEM_DEVICE) {
            d_t0 = t0_orbit;
        } else {
            CU(c, grow(c->d_t0, c->t0_cap, n));
            CU(c, cudaMemcpyAsync(c->d_t0, t0_orbit, (size_t)n * 8, cudaMemcpyDefault, c->stream));
            d_t0 = c->d_t0;
        }
    }
    if (n > c->acc_cap) {
        int64_t cap;
        cap = c->acc_cap; CU(c, grow(c->d_S, cap, n));
        cap = c->acc_cap; CU(c, grow(c->d_Wt, cap, n));
        cap = c->acc_cap; CU(c, grow(c->d_snr, cap, n));
        cap = c->acc_cap; CU(c, grow(c->d_cnt, cap, n));
        cap = c->acc_cap; CU(c, grow(c->d_hits, cap, n));
        c->acc_cap = n;
    }
    // sky order: kernels 1 and 3 work on a sorted copy of every unit, the sums come back in the caller's order
    const bool sorted = c->sort_orbits != 0;
    double *acc_S = c->d_S, *acc_Wt = c->d_Wt;
    int32_t *acc_cnt = c->d_cnt;
    if (sorted) {
        CU(c, grow(c->d_els, c->els_cap, n * 6));
        if (d_t0) CU(c, grow(c->d_t0s, c->t0s_cap, n));
        CU(c, grow(c->d_Ss, c->Ss_cap, n));
        CU(c, grow(c->d_Wts, c->Wts_cap, n));
        CU(c, grow(c->d_cnts, c->cnts_cap, n));
        CU(c, grow(c->d_perm, c->perm_cap, n));
        CU(c, grow(c->d_skey, c->skey_cap, 3 * unit_orb));
        const size_t need = sky_sort_temp_bytes(unit_orb);
        if (need > c->sort_tmp_bytes) {
            cudaFree(c->d_sort_tmp);
            c->d_sort_tmp = nullptr;
            c->sort_tmp_bytes = 0;
            CU(c, cudaMalloc(&c->d_sort_tmp, need));
            c->sort_tmp_bytes = need;
        }
        acc_S = c->d_Ss;
        acc_Wt = c->d_Wts;
        acc_cnt = c->d_cnts;
    }
    CU(c, grow(c->d_mask, c->mask_cap, unit_orb * unit_groups));
    CU(c, grow(c->d_base, c->base_cap, (unit_orb / 32) * unit_groups));
    CU(c, grow(c->d_offsets, c->off_cap, unit_orb * (int64_t)unit_groups * kGroup));
    while ((int64_t)c->ev_pool.size() < 4) {
        cudaEvent_t e;
        CU(c, cudaEventCreate(&e));
        c->ev_pool.push_back(e);
    }
    auto ev_at = [&](int i) { return c->ev_pool[4 + i]; };
    int unit_idx = 0;

    CU(c, cudaEventRecord(c->ev_pool[0], c->stream));
    CU(c, cudaMemsetAsync(acc_S, 0, (size_t)n * 8, c->stream));
    CU(c, cudaMemsetAsync(acc_Wt, 0, (size_t)n * 8, c->stream));
    CU(c, cudaMemsetAsync(acc_cnt, 0, (size_t)n * 4, c->stream));
    CU(c, reset_counters(c));

    const int mode = propagate_mode(c);
    int32_t k1_launches = 0;        // kernels enqueued for kernel 1: one per unit, or both variants + the policy update

    auto issue_copy = [&](int b) -> int {
        const int slot = b & 1;
        const int32_t first = b * unit_exp, cnt = std::min<int32_t>(unit_exp, c->N - first);
        if (c->ev_free_recorded[slot]) CU(c, cudaStreamWaitEvent(c->copy_stream, c->ev_free[slot], 0));
        for (int32_t j = 0; j < cnt; ++j) {
            CU(c, cudaMemcpyAsync(c->d_buf_flux[slot] + (int64_t)j * c->plane, c->h_flux[first + j],
                                  (size_t)c->plane * 4, cudaMemcpyHostToDevice, c->copy_stream));
            st.h2d_image_bytes += c->plane * 4;
            if (c->var_mode == 1) {
                CU(c, cudaMemcpyAsync(c->d_buf_var[slot] + (int64_t)j * c->plane, c->h_var[first + j],
                                      (size_t)c->plane * 4, cudaMemcpyHostToDevice, c->copy_stream));
                st.h2d_image_bytes += c->plane * 4;
            }
        }
        CU(c, cudaEventRecord(c->ev_ready[slot], c->copy_stream));
        return DT_OK;
    };

    // ---- streaming mode, few hits: gather straight from the page-locked host planes (zero-copy) ----
    // A survey larger than HBM costs its whole size over PCIe per pass when it is streamed (268 GB at
    // 55 GB/s = 4.9 s on configs[2]) although a blind search touches a few pixels per exposure (the
    // paper's own observation, "extremely sparse").  When the planes are device-mappable
    // and a probe (kernel 1 on the first orbit unit and exposure batch) predicts that the gathers
    // would move less than 5 % of the bytes streaming would, no image is copied at all and the sparse
    // gather reads the hit pixels over PCIe.  Same pixels, same arithmetic: bit-identical results.
    bool zero_copy_images = false;
    bool mappable = false;
    if (c->streaming && (c->stream_zero_copy != 0 || c->stream_tiles != 0)) {
        std::vector<const float *> hf(c->N), hv(c->N, nullptr);
        mappable = true;
        for (int32_t j = 0; j < c->N && mappable; ++j) {
            void *d = nullptr;
            mappable = cudaHostGetDevicePointer(&d, const_cast<float *>(c->h_flux[j]), 0) == cudaSuccess && d;
            hf[j] = static_cast<const float *>(d);
            if (mappable && c->var_mode == 1) {
                mappable = cudaHostGetDevicePointer(&d, const_cast<float *>(c->h_var[j]), 0) == cudaSuccess && d;
                hv[j] = static_cast<const float *>(d);
            }
        }
        if (!mappable) {
            cudaGetLastError();
        } else {
            if (!c->d_flux_ptrs) CU(c, cudaMalloc((void **)&c->d_flux_ptrs, sizeof(float *) * (size_t)c->N));
            if (!c->d_var_ptrs) CU(c, cudaMalloc((void **)&c->d_var_ptrs, sizeof(float *) * (size_t)c->N));
            CU(c, cudaMemcpyAsync((void *)c->d_flux_ptrs, hf.data(), sizeof(float *) * (size_t)c->N,
                                  cudaMemcpyHostToDevice, c->stream));
            CU(c, cudaMemcpyAsync((void *)c->d_var_ptrs, hv.data(), sizeof(float *) * (size_t)c->N,
                                  cudaMemcpyHostToDevice, c->stream));
            if (c->stream_zero_copy == 1) {
                zero_copy_images = true;
            } else if (c->stream_zero_copy != 0) {
                const int64_t no = std::min<int64_t>(unit_orb, n);
                const int32_t ne = std::min<int32_t>(unit_exp_max, c->N);
                PropagateParams p;
                fill_common(c, p, t0);
                if (elements_by_unit) CU(c, cudaStreamWaitEvent(c->stream, c->ev_elem[0], 0));
                p.elements = first_src;
                p.t0_orbit = d_t0;
                p.n_orbits = no;
                p.n_pad = (no + 31) / 32 * 32;
                p.exp = c->d_exp;
                p.n_exp = ne;
                p.groups_per_split = pick_groups_per_split(no, ne);
                p.mask = c->d_mask;
                p.base = c->d_base;
                p.offsets = c->d_offsets;
                p.counters = c->d_counters;
                CU(c, launch_k1_unit(c, p, mode, &k1_launches));
                st.propagate_launches += 1;
                unsigned long long probe_hits = 0;
                CU(c, cudaMemcpyAsync(&probe_hits, c->d_counters, sizeof probe_hits, cudaMemcpyDeviceToHost, c->stream));
                CU(c, cudaStreamSynchronize(c->stream));
                CU(c, reset_counters(c));
                const double planes = (c->var_mode == 1) ? 2.0 : 1.0;
                const double gathers = (double)probe_hits / ((double)no * ne) * (double)n * c->N * planes;
                zero_copy_images = gathers * 128.0 < 0.05 * (double)c->N * (double)c->plane * 4.0 * planes;
            }
        }
    }
    st.image_zero_copy = zero_copy_images ? 1 : 0;

    // ---- streaming mode, many hits: hits first, then only the image TILES the hits fall on cross PCIe, into a
    // device tile cache (dt_tiles.cu; PAPER.md:192 tiled layout, PAPER.md:330-332 pipelining); whole-plane double
    // buffering remains for planes that are not device-mappable or when the cache is switched off ----
    bool tiled = false;
    if (c->streaming && !zero_copy_images) {
        if (mappable && c->stream_tiles != 0) {
            rc = ensure_tile_cache(c);
            if (rc != DT_OK) return rc;
            tiled = true;
            CU(c, cudaMemsetAsync(c->tile_alloc, 0, 8 * sizeof(unsigned int), c->stream));
        } else {
            rc = ensure_stream_slots(c);
            if (rc != DT_OK) return rc;
            unit_exp = c->batch_exp;
        }
    }
    st.image_tiles = tiled ? 1 : 0;
    const int n_batches = (c->N + unit_exp - 1) / unit_exp;
    st.n_image_batches = n_batches;
    {
        const int64_t n_units_total = (int64_t)n_batches * ((n + unit_orb - 1) / unit_orb);
        while ((int64_t)c->ev_pool.size() < 4 + 3 * n_units_total) {
            cudaEvent_t e;
            CU(c, cudaEventCreate(&e));
            c->ev_pool.push_back(e);
        }
    }

    if (c->streaming && !zero_copy_images && !tiled) {
        // the copy stream must not start before earlier work on the context stream that may still
        // read the slots (a previous dt_stack) has been ordered: previous calls synchronise, so
        // only the free events of this call matter
        c->ev_free_recorded[0] = c->ev_free_recorded[1] = false;
        rc = issue_copy(0);
        if (rc != DT_OK) return rc;
    }

    for (int b = 0; b < n_batches; ++b) {
        const int slot = b & 1;
        const int32_t first = b * unit_exp, n_exp = std::min<int32_t>(unit_exp, c->N - first);
        if (c->streaming && !zero_copy_images && !tiled && b + 1 < n_batches) {
            rc = issue_copy(b + 1);
            if (rc != DT_OK) return rc;
        }
        if (tiled) {       // a fresh cache for this exposure unit: no tile resident, no slot handed out
            CU(c, cudaMemsetAsync(c->tile_slot, 0xff, (size_t)n_exp * (size_t)c->tiles_per_plane * sizeof(int32_t), c->stream));
            CU(c, cudaMemsetAsync(c->tile_alloc, 0, sizeof(unsigned int), c->stream));
        }
        bool waited = false;
        for (int64_t o0 = 0; o0 < n; o0 += unit_orb) {
            const int64_t no = std::min<int64_t>(unit_orb, n - o0);
            PropagateParams p;
            fill_common(c, p, t0);
            p.elements = (b == 0 ? first_src : d_el) + o0 * 6;
            p.t0_orbit = d_t0 ? d_t0 + o0 : nullptr;
            p.elements_copy = (b == 0 && copy_out) ? copy_out + o0 * 6 : nullptr;
            if (b == 0 && elements_by_unit) CU(c, cudaStreamWaitEvent(c->stream, c->ev_elem[o0 / unit_orb], 0));
            CU(c, cudaEventRecord(ev_at(3 * unit_idx), c->stream));
            if (sorted) {
                if (b == 0)       // once per orbit unit: the order of the survey's middle exposure serves every batch
                    CU(c, sky_sort_unit(d_el + o0 * 6, d_t0 ? d_t0 + o0 : nullptr, no, t0, c->d_exp + c->N / 2, c->gm,
                                        c->cos_eps, c->sin_eps, c->d_skey, c->d_skey + unit_orb, c->d_skey + 2 * unit_orb,
                                        c->d_sort_tmp, c->sort_tmp_bytes, c->d_perm + o0, c->d_els + o0 * 6,
                                        c->d_t0s + (d_t0 ? o0 : 0), c->stream));
                p.elements = c->d_els + o0 * 6;
                p.t0_orbit = d_t0 ? c->d_t0s + o0 : nullptr;
                p.elements_copy = nullptr;
            }
            p.n_orbits = no;
            p.n_pad = (no + 31) / 32 * 32;
            p.exp = c->d_exp + first;
            p.n_exp = n_exp;
            p.groups_per_split = pick_groups_per_split(no, n_exp);
            p.mask = c->d_mask;
            p.base = c->d_base;
            p.offsets = c->d_offsets;
            p.counters = c->d_counters;
            // the hit counter restarts per unit so offsets index from 0
            CU(c, cudaMemsetAsync(c->d_counters, 0, sizeof(unsigned long long), c->stream));
            CU(c, launch_k1_unit(c, p, mode, &k1_launches));
            st.propagate_launches += 1;
            CU(c, cudaEventRecord(ev_at(3 * unit_idx + 1), c->stream));

            if (c->streaming && !zero_copy_images && !tiled && !waited) {
                CU(c, cudaStreamWaitEvent(c->stream, c->ev_ready[slot], 0));
                waited = true;
            }
            GatherParams g;
            memset(&g, 0, sizeof g);
            if (tiled) {
                TileParams t;
                memset(&t, 0, sizeof t);
                t.n_pad = p.n_pad;
                t.n_groups = (n_exp + kGroup - 1) / kGroup;
                t.mask = c->d_mask;
                t.base = c->d_base;
                t.offsets = c->d_offsets;
                t.n_exp = n_exp;
                t.first_exposure = first;
                t.width = c->W;
                t.height = c->H;
                t.ts_log2 = kTileLog2;
                t.tiles_x = c->tiles_x;
                t.tiles_per_plane = c->tiles_per_plane;
                t.tile_count = c->tile_count;
                t.tile_slot = c->tile_slot;
                t.alloc = c->tile_alloc;
                t.capacity = c->tile_capacity;
                // default: a tile is worth its transfer from 32 hits on (a 32-KB tile of flux + variance: 1 KB per hit; measured on
                // lsst+focused: kernel 3 74 ms per step at 128 hits, 55 ms at 32 and at 8, 1.2 / 1.5 / 1.7 GB over PCIe)
                t.min_hits = c->tile_min_hits > 0 ? c->tile_min_hits : (int32_t)std::max<int64_t>(1, c->slot_floats * 4 / 1024);
                t.fetch_list = c->tile_fetch;
                t.flux_ptrs = c->d_flux_ptrs;
                t.var_ptrs = (c->var_mode == 1) ? c->d_var_ptrs : nullptr;
                t.tile_buf = c->tile_buf;
                t.slot_floats = c->slot_floats;
                t.offsets_cap = c->off_cap;
                t.bounds = c->d_counters + 7;
                CU(c, launch_tiles(t, c->sm_count, c->stream));
                g.tile_slot = c->tile_slot;
                g.tile_buf = c->tile_buf;
                g.slot_floats = c->slot_floats;
                g.ts_log2 = kTileLog2;
                g.tiles_x = c->tiles_x;
                g.tiles_per_plane = c->tiles_per_plane;
                g.tile_e0 = first;
            }
            g.n_orbits = no;
            g.n_pad = p.n_pad;
            g.first_exposure = first;
            g.n_groups = (n_exp + kGroup - 1) / kGroup;
            g.mask = c->d_mask;
            g.base = c->d_base;
            g.offsets = c->d_offsets;
            if (zero_copy_images || tiled) {
                g.flux_ptrs = c->d_flux_ptrs;
                g.var_ptrs = (c->var_mode == 1) ? c->d_var_ptrs : nullptr;
            } else if (c->streaming) {
                g.flux = c->d_buf_flux[slot] - (int64_t)first * c->plane;
                g.var = (c->var_mode == 1) ? c->d_buf_var[slot] - (int64_t)first * c->plane : nullptr;
            } else {
                g.flux = c->d_flux;              // scalar-variance mode
                g.fv = c->d_fv;                  // plane-variance mode (one of the two is NULL)
            }
            g.exp_all = c->d_exp;
            g.plane = c->plane;
            g.S = acc_S + o0;
            g.Wt = acc_Wt + o0;
            g.cnt = acc_cnt + o0;
            g.progress = c->d_progress;
            g.window = c->gather_window;
            g.n_hits_dev = c->d_counters;            // the unit's hit allocator, final after kernel 1
            g.lockstep_mode = (zero_copy_images || tiled) ? 0 : c->gather_lockstep;
            g.ld_cached = c->gather_ld_cached;
            g.prefetch = c->streaming ? 0 : c->gather_prefetch;
            g.n_exp_store = c->N;
            g.sm_count = c->sm_count;
            fill_gather_ext(c, g);
            CU(c, launch_gather_unit(c, g, &st.gather_launches));
            CU(c, cudaEventRecord(ev_at(3 * unit_idx + 2), c->stream));
            unit_idx += 1;
        }
        if (c->streaming && !zero_copy_images && !tiled) {
            CU(c, cudaEventRecord(c->ev_free[slot], c->stream));
            c->ev_free_recorded[slot] = true;
        }
    }
    CU(c, cudaEventRecord(c->ev_pool[2], c->stream));
    if (sorted)
        CU(c, sky_unsort_sums(c->d_perm, n, unit_orb, c->d_Ss, c->d_Wts, c->d_cnts, c->d_S, c->d_Wt, c->d_cnt, c->stream));
    CU(c, launch_finalize(d_el, d_t0, n, c->d_S, c->d_Wt, c->d_cnt, c->d_snr, c->d_hits, c->d_counters + 5,
                          c->stream));
    CU(c, cudaEventRecord(c->ev_pool[3], c->stream));
    if (snr_out)
        CU(c, cudaMemcpyAsync(snr_out, c->d_snr, (size_t)n * 8, cudaMemcpyDefault, c->stream));
    if (hits_out)
        CU(c, cudaMemcpyAsync(hits_out, c->d_hits, (size_t)n * 4, cudaMemcpyDefault, c->stream));
    CU(c, cudaEventRecord(c->ev_pool[1], c->stream));
    unsigned long long hc[8];
    unsigned int tc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    CU(c, cudaMemcpyAsync(hc, c->d_counters, sizeof hc, cudaMemcpyDeviceToHost, c->stream));
    if (tiled) CU(c, cudaMemcpyAsync(tc, c->tile_alloc, sizeof tc, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    st.tiles_fetched = (int64_t)tc[2];
    st.h2d_image_bytes += (int64_t)tc[2] * c->slot_floats * 4;
    CU(c, cudaEventElapsedTime(&st.ms_total, c->ev_pool[0], c->ev_pool[1]));
    CU(c, cudaEventElapsedTime(&st.ms_finalize, c->ev_pool[2], c->ev_pool[3]));
    for (int u = 0; u < unit_idx; ++u) {
        float a = 0.f, b = 0.f;
        CU(c, cudaEventElapsedTime(&a, ev_at(3 * u), ev_at(3 * u + 1)));
        CU(c, cudaEventElapsedTime(&b, ev_at(3 * u + 1), ev_at(3 * u + 2)));
        st.ms_propagate += a;
        st.ms_gather += b;
    }
    st.hits = (int64_t)hc[3];
    st.refined_pairs = (int64_t)hc[1];
    st.cold_solves = (int64_t)hc[2];
    st.substep_solves = (int64_t)hc[4];
    st.invalid_orbits = (int64_t)hc[5];
    st.gated_pairs = (int64_t)hc[6];
    if (hc[7] != 0)
        return fail(c, DT_ERR_CUDA, "bounds-check build: %llu out-of-bounds indices were caught on the device", hc[7]);
    st.launches = k1_launches + st.gather_launches + 1;
    c->n_last = n;
    return DT_OK;
}

extern "C" {

int dt_stack(dt_context *c, const double *elements, int64_t n, double t0, int32_t mem_kind, double *snr_out,
             int32_t *hits_out)
{
    return stack_impl(c, elements, nullptr, n, t0, mem_kind, snr_out, hits_out);
}

int dt_stack_epochs(dt_context *c, const double *elements, const double *t0, int64_t n, int32_t mem_kind,
                    double *snr_out, int32_t *hits_out)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (n > 0 && !t0) return fail(c, DT_ERR_INVALID_ARG, "dt_stack_epochs: t0 is NULL");
    return stack_impl(c, elements, n > 0 ? t0 : nullptr, n, 0.0, mem_kind, snr_out, hits_out);
}

int dt_set_patch(dt_context *c, int32_t k, const double *weights)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (k < 1 || k > 15 || (k % 2) == 0) return fail(c, DT_ERR_INVALID_ARG, "dt_set_patch: k must be odd, 1 .. 15");
    if (weights)
        for (int i = 0; i < k * k; ++i)
            if (!isfinite(weights[i])) return fail(c, DT_ERR_INVALID_ARG, "dt_set_patch: non-finite weight");
    CU(c, cudaSetDevice(c->device));
    CU(c, cudaStreamSynchronize(c->stream));
    cudaFree(c->d_patch_w);
    c->d_patch_w = nullptr;
    c->patch = k;
    if (weights) {
        CU(c, cudaMalloc((void **)&c->d_patch_w, sizeof(double) * (size_t)(k * k)));
        CU(c, cudaMemcpy(c->d_patch_w, weights, sizeof(double) * (size_t)(k * k), cudaMemcpyHostToDevice));
    }
    return DT_OK;
}

int dt_set_outlier_clip(dt_context *c, double clip)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (isnan(clip)) return fail(c, DT_ERR_INVALID_ARG, "dt_set_outlier_clip: NaN");
    c->clip = clip;
    return DT_OK;
}

int dt_threshold(dt_context *c, double snr_min, int32_t min_hits, int64_t max_out, int64_t *index_out,
                 double *snr_out, int64_t *n_found)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (isnan(snr_min) || max_out < 0 || !n_found || (max_out > 0 && !index_out))
        return fail(c, DT_ERR_INVALID_ARG, "dt_threshold: bad arguments");
    if (c->n_last < 0) return fail(c, DT_ERR_STATE, "dt_threshold: no dt_stack result on the device");
    CU(c, cudaSetDevice(c->device));
    CU(c, threshold_device(c->d_snr, c->d_hits, c->n_last, snr_min, min_hits, max_out, c->topk, index_out, snr_out,
                           n_found, c->stream));
    return DT_OK;
}

int dt_threshold_noalloc(void *stream, const double *snr_dev, const int32_t *hits_dev, int64_t n, double snr_min,
                         int32_t min_hits, int64_t max_out, int64_t *index_out_dev, double *snr_out_dev,
                         int64_t *n_found_dev)
{
    if (n < 0 || max_out < 0 || isnan(snr_min) || !n_found_dev || (n > 0 && (!snr_dev || !hits_dev)) ||
        (n > 0 && max_out > 0 && !index_out_dev)) {
        g_static_err = "dt_threshold_noalloc: bad arguments";
        return DT_ERR_INVALID_ARG;
    }
    if (n > threshold_noalloc_max()) {
        g_static_err = "dt_threshold_noalloc: n exceeds DT_NOALLOC_MAX_ORBITS (1048576), the size the library's static "
                       "scratch array is built for; split the array or use dt_threshold";
        return DT_ERR_TOO_LARGE;
    }
    static_assert(sizeof(long long) == sizeof(int64_t), "int64");
    const cudaError_t e = threshold_noalloc_device(snr_dev, hits_dev, n, snr_min, min_hits, max_out,
                                                   reinterpret_cast<long long *>(index_out_dev), snr_out_dev,
                                                   reinterpret_cast<long long *>(n_found_dev), (cudaStream_t)stream);
    if (e != cudaSuccess) {
        g_static_err = cudaGetErrorString(e);
        return DT_ERR_CUDA;
    }
    return DT_OK;
}

static int partial_scratch(dt_context *c, int64_t m)
{
    if (m <= c->p_cap && c->d_pidx) return DT_OK;
    cudaFree(c->d_pidx); cudaFree(c->d_pS); cudaFree(c->d_pW); cudaFree(c->d_pc);
    c->d_pidx = nullptr; c->d_pS = c->d_pW = nullptr; c->d_pc = nullptr; c->p_cap = 0;
    const size_t k = (size_t)std::max<int64_t>(m, 1);
    CU(c, cudaMalloc((void **)&c->d_pidx, k * 8));
    CU(c, cudaMalloc((void **)&c->d_pS, k * 8));
    CU(c, cudaMalloc((void **)&c->d_pW, k * 8));
    CU(c, cudaMalloc((void **)&c->d_pc, k * 4));
    c->p_cap = (int64_t)k;
    return DT_OK;
}

int dt_partials_sparse(dt_context *c, int64_t max_out, int64_t *index_out, double *S_out, double *Wt_out,
                       int32_t *cnt_out, int32_t mem_kind, int64_t *n_found)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (max_out < 0 || !n_found || !mem_kind_ok(mem_kind) || (max_out > 0 && (!index_out || !S_out || !Wt_out || !cnt_out)))
        return fail(c, DT_ERR_INVALID_ARG, "dt_partials_sparse: bad arguments");
    if (c->n_last < 0) return fail(c, DT_ERR_STATE, "dt_partials_sparse: no dt_stack result on the device");
    CU(c, cudaSetDevice(c->device));
    const int64_t n = c->n_last, cap = std::min<int64_t>(max_out, n);
    long long *di = reinterpret_cast<long long *>(index_out);
    double *dS = S_out, *dW = Wt_out;
    int32_t *dc = cnt_out;
    if (mem_kind != DT_MEM_DEVICE) {
        int rc = partial_scratch(c, cap);
        if (rc != DT_OK) return rc;
        di = c->d_pidx; dS = c->d_pS; dW = c->d_pW; dc = c->d_pc;
    }
    CU(c, partials_sparse_device(c->d_S, c->d_Wt, c->d_cnt, n, cap, c->topk, di, dS, dW, dc, n_found, c->stream));
    const int64_t m = std::min<int64_t>(*n_found, cap);
    if (mem_kind != DT_MEM_DEVICE && m > 0) {
        CU(c, cudaMemcpyAsync(index_out, di, (size_t)m * 8, cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaMemcpyAsync(S_out, dS, (size_t)m * 8, cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaMemcpyAsync(Wt_out, dW, (size_t)m * 8, cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaMemcpyAsync(cnt_out, dc, (size_t)m * 4, cudaMemcpyDeviceToHost, c->stream));
    }
    CU(c, cudaStreamSynchronize(c->stream));
    return DT_OK;
}

int dt_partials_reset(dt_context *c)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (c->n_last < 0) return fail(c, DT_ERR_STATE, "dt_partials_reset: no dt_stack result on the device");
    CU(c, cudaSetDevice(c->device));
    const size_t n = (size_t)c->n_last;
    CU(c, cudaMemsetAsync(c->d_S, 0, n * 8, c->stream));
    CU(c, cudaMemsetAsync(c->d_Wt, 0, n * 8, c->stream));
    CU(c, cudaMemsetAsync(c->d_cnt, 0, n * 4, c->stream));
    return DT_OK;
}

int dt_partials_add(dt_context *c, const int64_t *index, const double *S, const double *Wt, const int32_t *cnt,
                    int64_t m, int32_t mem_kind)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (m < 0 || !mem_kind_ok(mem_kind) || (m > 0 && (!index || !S || !Wt || !cnt)))
        return fail(c, DT_ERR_INVALID_ARG, "dt_partials_add: bad arguments");
    if (c->n_last < 0) return fail(c, DT_ERR_STATE, "dt_partials_add: no dt_stack result on the device");
    if (m == 0) return DT_OK;
    CU(c, cudaSetDevice(c->device));
    const long long *di = reinterpret_cast<const long long *>(index);
    const double *dS = S, *dW = Wt;
    const int32_t *dc = cnt;
    if (mem_kind != DT_MEM_DEVICE) {
        int rc = partial_scratch(c, m);
        if (rc != DT_OK) return rc;
        CU(c, cudaMemcpyAsync(c->d_pidx, index, (size_t)m * 8, cudaMemcpyDefault, c->stream));
        CU(c, cudaMemcpyAsync(c->d_pS, S, (size_t)m * 8, cudaMemcpyDefault, c->stream));
        CU(c, cudaMemcpyAsync(c->d_pW, Wt, (size_t)m * 8, cudaMemcpyDefault, c->stream));
        CU(c, cudaMemcpyAsync(c->d_pc, cnt, (size_t)m * 4, cudaMemcpyDefault, c->stream));
        di = c->d_pidx; dS = c->d_pS; dW = c->d_pW; dc = c->d_pc;
    }
    if (!c->d_bad) CU(c, cudaMalloc((void **)&c->d_bad, sizeof(int)));
    CU(c, cudaMemsetAsync(c->d_bad, 0, sizeof(int), c->stream));
    CU(c, partials_add_device(di, m, c->n_last, dS, dW, dc, c->d_S, c->d_Wt, c->d_cnt, c->d_bad, c->stream));
    int bad = 0;
    CU(c, cudaMemcpyAsync(&bad, c->d_bad, sizeof bad, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    if (bad) return fail(c, DT_ERR_INVALID_ARG, "dt_partials_add: an orbit index is outside [0, n)");
    return DT_OK;
}

int dt_partials_finalize(dt_context *c, double *snr_out, int32_t *hits_out, int32_t mem_kind)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (!mem_kind_ok(mem_kind)) return fail(c, DT_ERR_INVALID_ARG, "dt_partials_finalize: bad arguments");
    if (c->n_last < 0) return fail(c, DT_ERR_STATE, "dt_partials_finalize: no dt_stack result on the device");
    CU(c, cudaSetDevice(c->device));
    const int64_t n = c->n_last;
    CU(c, refinalize_device(n, c->d_S, c->d_Wt, c->d_cnt, c->d_snr, c->d_hits, c->stream));
    if (snr_out) CU(c, cudaMemcpyAsync(snr_out, c->d_snr, (size_t)n * 8, cudaMemcpyDefault, c->stream));
    if (hits_out) CU(c, cudaMemcpyAsync(hits_out, c->d_hits, (size_t)n * 4, cudaMemcpyDefault, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return DT_OK;
}

int dt_topk(dt_context *c, int32_t k, int32_t min_hits, int64_t *index_out, double *snr_out, int32_t *n_found)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (k < 0 || !n_found || (k > 0 && (!index_out || !snr_out)))
        return fail(c, DT_ERR_INVALID_ARG, "dt_topk: bad arguments");
    if (c->n_last < 0) return fail(c, DT_ERR_STATE, "dt_topk: no dt_stack result on the device");
    CU(c, cudaSetDevice(c->device));
    CU(c, topk_device(c->d_snr, c->d_hits, c->n_last, k, min_hits, c->topk, index_out, snr_out, n_found,
                      c->stream));
    return DT_OK;
}

int dt_project(dt_context *c, const double *elements, int64_t n, double t0, double *radec_out, double *xy_out,
               int32_t *pix_out)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (n < 0 || (n > 0 && !elements) || !isfinite(t0)) return fail(c, DT_ERR_INVALID_ARG, "dt_project: bad arguments");
    if (n == 0) return DT_OK;
    CU(c, cudaSetDevice(c->device));
    const int64_t N = c->N;
    int64_t chunk = std::max<int64_t>(32, (int64_t)(6400000 / N) / 32 * 32);
    chunk = std::min<int64_t>(chunk, (n + 31) / 32 * 32);
    double *d_el = nullptr, *d_radec = nullptr, *d_xy = nullptr;
    int32_t *d_pix = nullptr;
    int rc = DT_OK;
    auto cleanup = [&]() {
        cudaFree(d_el);
        cudaFree(d_radec);
        cudaFree(d_xy);
        cudaFree(d_pix);
    };
#define CUP(call)                                                                                 \
    do {                                                                                          \
        cudaError_t e__ = (call);                                                                 \
        if (e__ != cudaSuccess) {                                                                 \
            cleanup();                                                                            \
            return fail(c, DT_ERR_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__));         \
        }                                                                                         \
    } while (0)
    CUP(cudaMalloc((void **)&d_el, (size_t)chunk * 48));
    CUP(cudaMalloc((void **)&d_radec, (size_t)chunk * N * 16));
    CUP(cudaMalloc((void **)&d_xy, (size_t)chunk * N * 16));
    CUP(cudaMalloc((void **)&d_pix, (size_t)chunk * N * 8));
    // default: every pair refined; DT_FLAG_PROJECT_PRECULL keeps dt_stack's pre-cull and cull-quality chain, and the
    // group ephemeris gate unless it is switched off (no device-side choice here: a parity entry runs what it is told)
    int mode = propagate_mode(c) & (kModeWarm | ((c->flags & DT_FLAG_PROJECT_PRECULL) ? kModePrecull : 0));
    if (mode == (kModeWarm | kModePrecull) && !(c->flags & DT_FLAG_NO_GROUP_GATE) && c->group_gate != 0) mode |= kModeGate;
    mode |= kModeDense;
    for (int64_t o0 = 0; o0 < n; o0 += chunk) {
        const int64_t no = std::min<int64_t>(chunk, n - o0);
        CUP(cudaMemcpyAsync(d_el, elements + o0 * 6, (size_t)no * 48, cudaMemcpyHostToDevice, c->stream));
        PropagateParams p;
        fill_common(c, p, t0);
        p.elements = d_el;
        p.n_orbits = no;
        p.n_pad = (no + 31) / 32 * 32;
        p.exp = c->d_exp;
        p.n_exp = c->N;
        p.groups_per_split = pick_groups_per_split(no, c->N);
        p.counters = c->d_counters;
        p.radec = d_radec;
        p.xy = d_xy;
        p.pix = d_pix;
        CUP(launch_propagate(p, mode, c->stream));
        if (radec_out)
            CUP(cudaMemcpyAsync(radec_out + o0 * N * 2, d_radec, (size_t)no * N * 16, cudaMemcpyDeviceToHost, c->stream));
        if (xy_out)
            CUP(cudaMemcpyAsync(xy_out + o0 * N * 2, d_xy, (size_t)no * N * 16, cudaMemcpyDeviceToHost, c->stream));
        if (pix_out)
            CUP(cudaMemcpyAsync(pix_out + o0 * N * 2, d_pix, (size_t)no * N * 8, cudaMemcpyDeviceToHost, c->stream));
        CUP(cudaStreamSynchronize(c->stream));
    }
#undef CUP
    cleanup();
    return rc;
}

int dt_gather_hits(dt_context *c, int64_t n, int32_t first_exposure, int32_t n_groups, const uint32_t *mask,
                   const uint64_t *base, const uint32_t *offsets, int64_t n_hits, double *S, double *Wt, int32_t *cnt)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (n < 0 || n_hits < 0 || n_hits >= ((int64_t)1 << 32) || n_groups < 0 || first_exposure < 0 || (int64_t)first_exposure + (int64_t)n_groups * kGroup > (c->N + kGroup - 1) / kGroup * kGroup ||
        !mask || !base || !offsets || !S || !Wt || !cnt)
        return fail(c, DT_ERR_INVALID_ARG, "dt_gather_hits: bad arguments");
    if (n > kMaxUnitOrbits || n_groups > kMaxUnitExposures / kGroup)
        return fail(c, DT_ERR_INVALID_ARG, "dt_gather_hits: at most %lld orbits and %d groups per call",
                    (long long)kMaxUnitOrbits, kMaxUnitExposures / kGroup);
    if (c->streaming || (!c->d_flux && !c->d_fv)) return fail(c, DT_ERR_STATE, "dt_gather_hits needs resident images");
    CU(c, cudaSetDevice(c->device));
    GatherParams g;
    memset(&g, 0, sizeof g);
    g.n_orbits = n;
    g.n_pad = (n + 31) / 32 * 32;
    g.first_exposure = first_exposure;
    g.n_groups = n_groups;
    g.mask = mask;
    g.base = (const unsigned long long *)base;
    g.offsets = offsets;
    g.flux = c->d_flux;
    g.fv = c->d_fv;
    g.exp_all = c->d_exp;
    g.plane = c->plane;
    g.S = S;
    g.Wt = Wt;
    g.cnt = cnt;
    g.progress = c->d_progress;
    g.window = c->gather_window;
    g.n_hits_dev = nullptr;
    g.n_hits_host = n_hits;
    g.lockstep_mode = c->gather_lockstep;
    g.ld_cached = c->gather_ld_cached;
    g.prefetch = c->gather_prefetch;
    g.n_exp_store = c->N;
    g.sm_count = c->sm_count;
    fill_gather_ext(c, g);
    g.offsets_cap = n_hits;
#ifdef DT_BOUNDS_CHECK
    CU(c, cudaMemsetAsync(c->d_counters + 7, 0, sizeof(unsigned long long), c->stream));
#endif
    {
        int32_t launches = 0;
        CU(c, launch_gather_unit(c, g, &launches));
    }
#ifdef DT_BOUNDS_CHECK
    {
        unsigned long long bad = 0;
        CU(c, cudaMemcpyAsync(&bad, c->d_counters + 7, sizeof bad, cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        if (bad) return fail(c, DT_ERR_CUDA, "bounds-check build: %llu out-of-bounds indices were caught on the device", bad);
    }
#endif
    return DT_OK;
}

int dt_filter_intersections(dt_context *c, const double *elements, int64_t n, double t0, int32_t mem_kind,
                            int32_t first_exposure, int32_t n_exposures, const uint32_t **mask,
                            const uint64_t **base, const uint32_t **offsets, int64_t *n_hits, int64_t *n_pad,
                            int32_t *n_groups)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (n < 1 || n > kMaxUnitOrbits || !elements || !mem_kind_ok(mem_kind) || !isfinite(t0) || first_exposure < 0 ||
        n_exposures < 1 || n_exposures > kMaxUnitExposures || (int64_t)first_exposure + n_exposures > c->N ||
        !mask || !base || !offsets || !n_hits || !n_pad || !n_groups)
        return fail(c, DT_ERR_INVALID_ARG, "dt_filter_intersections: bad arguments (one work unit: <= %lld orbits, <= %d exposures)",
                    (long long)kMaxUnitOrbits, kMaxUnitExposures);
    CU(c, cudaSetDevice(c->device));
    const int64_t pad = (n + 31) / 32 * 32;
    const int32_t groups = (n_exposures + kGroup - 1) / kGroup;
    const double *d_el = elements;
    if (mem_kind != DT_MEM_DEVICE || (reinterpret_cast<uintptr_t>(elements) & 15u)) {
        CU(c, grow(c->d_el, c->el_cap, n * 6));
        CU(c, cudaMemcpyAsync(c->d_el, elements, (size_t)n * 48, cudaMemcpyDefault, c->stream));
        d_el = c->d_el;
    }
    CU(c, grow(c->d_mask, c->mask_cap, pad * groups));
    CU(c, grow(c->d_base, c->base_cap, (pad / 32) * groups));
    CU(c, grow(c->d_offsets, c->off_cap, pad * (int64_t)groups * kGroup));
    CU(c, reset_counters(c));
    PropagateParams p;
    fill_common(c, p, t0);
    p.elements = d_el;
    p.n_orbits = n;
    p.n_pad = pad;
    p.exp = c->d_exp + first_exposure;
    p.n_exp = n_exposures;
    p.groups_per_split = pick_groups_per_split(n, n_exposures);
    p.mask = c->d_mask;
    p.base = c->d_base;
    p.offsets = c->d_offsets;
    p.counters = c->d_counters;
    int32_t k1_launches = 0;
    CU(c, launch_k1_unit(c, p, propagate_mode(c), &k1_launches));
    unsigned long long h = 0;
    CU(c, cudaMemcpyAsync(&h, c->d_counters, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    c->n_last = -1;                       // the per-orbit results of an earlier dt_stack are gone
    *mask = c->d_mask;
    *base = reinterpret_cast<const uint64_t *>(c->d_base);
    *offsets = c->d_offsets;
    *n_hits = (int64_t)h;
    *n_pad = pad;
    *n_groups = groups;
    return DT_OK;
}

int dt_sky_order(dt_context *c, const double *elements_dev, const double *t0_orbit_dev, int64_t n, double t0,
                 uint32_t *perm_out_dev)
{
    if (!c) return DT_ERR_INVALID_ARG;
    if (n < 0 || n > kMaxUnitOrbits || (n > 0 && (!elements_dev || !perm_out_dev)))
        return fail(c, DT_ERR_INVALID_ARG, "dt_sky_order: one unit of at most %lld orbits, device arrays", (long long)kMaxUnitOrbits);
    if (n == 0) return DT_OK;
    CU(c, cudaSetDevice(c->device));
    CU(c, grow(c->d_skey, c->skey_cap, 3 * kMaxUnitOrbits));
    const size_t need = sky_sort_temp_bytes(kMaxUnitOrbits);
    if (need > c->sort_tmp_bytes) {
        cudaFree(c->d_sort_tmp);
        c->d_sort_tmp = nullptr;
        c->sort_tmp_bytes = 0;
        CU(c, cudaMalloc(&c->d_sort_tmp, need));
        c->sort_tmp_bytes = need;
    }
    CU(c, sky_sort_unit(elements_dev, t0_orbit_dev, n, t0, c->d_exp + c->N / 2, c->gm, c->cos_eps, c->sin_eps, c->d_skey,
                        c->d_skey + kMaxUnitOrbits, c->d_skey + 2 * kMaxUnitOrbits, c->d_sort_tmp, c->sort_tmp_bytes,
                        perm_out_dev, nullptr, nullptr, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return DT_OK;
}

int dt_set_option(dt_context *c, const char *name, int64_t value)
{
    if (!c || !name) return DT_ERR_INVALID_ARG;
    const std::string k(name);
    if (k == "gather_schedule") {
        if (value < -1 || value > 1) return fail(c, DT_ERR_INVALID_ARG, "gather_schedule: -1 auto, 0 orbit-major, 1 dense");
        c->gather_lockstep = (int32_t)value;
    } else if (k == "group_gate") {
        if (value < -1 || value > 1) return fail(c, DT_ERR_INVALID_ARG, "group_gate: -1 chosen on the device, 0 off, 1 on");
        c->group_gate = (int32_t)value;
    } else if (k == "sort_orbits") {
        c->sort_orbits = value ? 1 : 0;
    } else if (k == "gather_slab") {
        c->gather_slab = (int32_t)std::max<int64_t>(-1, std::min<int64_t>(value, 1 << 20));
    } else if (k == "gather_window") {
        c->gather_window = value > 0 ? (int32_t)std::min<int64_t>(value, 64) : pick_gather_window(c);
    } else if (k == "gather_prefetch") {
        c->gather_prefetch = (int32_t)std::max<int64_t>(0, std::min<int64_t>(value, 8));
    } else if (k == "gather_l1") {
        c->gather_ld_cached = value ? 1 : 0;
    } else if (k == "stream_tiles") {
        c->stream_tiles = value < 0 ? -1 : (value ? 1 : 0);
    } else if (k == "tile_min_hits") {
        c->tile_min_hits = (int32_t)std::max<int64_t>(0, std::min<int64_t>(value, 1 << 30));
    } else if (k == "stream_zero_copy") {
        c->stream_zero_copy = value < 0 ? -1 : (value ? 1 : 0);
    } else if (k == "zero_copy_elements") {
        c->zero_copy_elements = value != 0;
    } else {
        return fail(c, DT_ERR_INVALID_ARG, "dt_set_option: unknown option '%s'", name);
    }
    return DT_OK;
}

int dt_get_stats(const dt_context *c, dt_stats *out)
{
    if (!c || !out || out->struct_size != sizeof(dt_stats)) return DT_ERR_INVALID_ARG;
    *out = c->stats;
    return DT_OK;
}

int dt_fp64_peak(int32_t device, double *tflops)
{
    if (!tflops) return DT_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return DT_ERR_CUDA;
    }
    if (cudaSetDevice(device) != cudaSuccess) return DT_ERR_CUDA;
    return fp64_peak_device(tflops, nullptr) == cudaSuccess ? DT_OK : DT_ERR_CUDA;
}

int dt_probe_random_gather(int32_t device, int64_t buffer_bytes, int32_t hint64, double *gathers_per_s)
{
    if (!gathers_per_s || buffer_bytes < (1 << 20)) return DT_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return DT_ERR_CUDA;
    }
    if (cudaSetDevice(device) != cudaSuccess) return DT_ERR_CUDA;
    const cudaError_t e = random_gather_probe(buffer_bytes, hint64, gathers_per_s, nullptr);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return DT_ERR_OOM; }
    return e == cudaSuccess ? DT_OK : DT_ERR_CUDA;
}

}  // extern "C"
