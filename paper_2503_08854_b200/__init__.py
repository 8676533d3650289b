"""paper_2503_08854_b200 -- thin Python binding of the dtrack-b200 C ABI (include/dtrack.h).

Argument marshalling only: every step of the hot path (propagate, light-time, project, cull,
compact, gather, stack, top-k) runs in the library's sm_100a CUDA kernels.  There is NO CPU
fallback and this package never imports the CPU oracle: if `libdtrack.so` is missing and cannot be
built, importing `lib()` raises; on a box without a CUDA device `dt_create` raises DtError.

The functions carry the C names (`dt_create`, `dt_load_image_batch`, `dt_stack`, `dt_topk`,
`dt_project`, `dt_gather_hits`, `dt_get_stats`, `dt_destroy`, `dt_fp64_peak`); `Tracker` is a small
convenience wrapper around one context.  Arrays may be numpy arrays (host), torch CPU tensors
(pinned or pageable) or torch CUDA tensors; PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from typing import Optional

import numpy as np

from . import _build

DT_OK, DT_ERR_INVALID_ARG, DT_ERR_OOM, DT_ERR_CUDA, DT_ERR_NOT_LOADED, DT_ERR_STATE = 0, -1, -2, -3, -4, -5
DT_MEM_HOST, DT_MEM_PINNED, DT_MEM_DEVICE = 0, 1, 2
DT_FLAG_FORCE_STREAM, DT_FLAG_KEPLER_COLD, DT_FLAG_NO_PRECULL, DT_FLAG_PROJECT_PRECULL, DT_FLAG_NO_GROUP_GATE = 1, 2, 4, 8, 16
_ERR_NAMES = {-1: "DT_ERR_INVALID_ARG", -2: "DT_ERR_OOM", -3: "DT_ERR_CUDA", -4: "DT_ERR_NOT_LOADED",
              -5: "DT_ERR_STATE", -6: "DT_ERR_TOO_LARGE"}
DT_NOALLOC_MAX_ORBITS = 1 << 20

EXPORTS = ["dt_create", "dt_destroy", "dt_load_image_batch", "dt_stack", "dt_stack_epochs", "dt_set_patch",
           "dt_set_outlier_clip", "dt_threshold", "dt_threshold_noalloc", "dt_partials_sparse", "dt_partials_reset", "dt_partials_add",
           "dt_partials_finalize", "dt_topk", "dt_project",
           "dt_gather_hits", "dt_filter_intersections", "dt_sky_order", "dt_set_option", "dt_get_stats", "dt_last_error", "dt_version", "dt_fp64_peak", "dt_probe_random_gather"]


class DtError(RuntimeError):
    def __init__(self, code: int, msg: str = ""):
        self.code = code
        super().__init__("%s (%d)%s" % (_ERR_NAMES.get(code, "error"), code, (": " + msg) if msg else ""))


class dt_survey(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_exposures", C.c_int32), ("width", C.c_int32),
                ("height", C.c_int32), ("t", C.POINTER(C.c_double)), ("obs_ecl", C.POINTER(C.c_double)),
                ("ra0", C.POINTER(C.c_double)), ("dec0", C.POINTER(C.c_double)),
                ("pixel_scale", C.c_double), ("gm", C.c_double), ("c", C.c_double),
                ("obliquity", C.c_double), ("variance_mode", C.c_int32),
                ("var_scalar", C.POINTER(C.c_double)), ("device", C.c_int32), ("stream", C.c_void_p),
                ("hbm_budget_bytes", C.c_int64), ("flags", C.c_uint32)]


class dt_stats(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_orbits", C.c_int64), ("n_exposures", C.c_int64),
                ("pairs", C.c_int64), ("hits", C.c_int64), ("invalid_orbits", C.c_int64),
                ("refined_pairs", C.c_int64), ("cold_solves", C.c_int64),
                ("substep_solves", C.c_int64), ("h2d_image_bytes", C.c_int64), ("streamed", C.c_int32), ("n_image_batches", C.c_int32),
                ("ms_total", C.c_float), ("ms_propagate", C.c_float), ("ms_gather", C.c_float),
                ("ms_finalize", C.c_float), ("launches", C.c_int32), ("propagate_launches", C.c_int32),
                ("gather_launches", C.c_int32), ("image_zero_copy", C.c_int32), ("image_tiles", C.c_int32),
                ("tiles_fetched", C.c_int64), ("gated_pairs", C.c_int64)]


_lib = None


def lib():
    """The loaded C-ABI library; built in-tree with nvcc on first use.  Raises when unavailable."""
    global _lib
    if _lib is None:
        path = os.environ.get("DTRACK_LIB") or _build.build()   # DTRACK_LIB: a prebuilt library
        if not os.path.exists(path):
            raise RuntimeError("libdtrack.so is missing and could not be built; there is no CPU fallback")
        L = C.CDLL(path)
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int32)
        L.dt_create.argtypes = [C.POINTER(dt_survey), C.POINTER(vp)]
        L.dt_destroy.argtypes = [vp]
        L.dt_load_image_batch.argtypes = [vp, C.c_int32, C.c_int32, vp, vp, C.c_int32]
        L.dt_stack.argtypes = [vp, vp, C.c_int64, C.c_double, C.c_int32, vp, vp]
        L.dt_stack_epochs.argtypes = [vp, vp, vp, C.c_int64, C.c_int32, vp, vp]
        L.dt_set_patch.argtypes = [vp, C.c_int32, dp]
        L.dt_set_outlier_clip.argtypes = [vp, C.c_double]
        L.dt_threshold.argtypes = [vp, C.c_double, C.c_int32, C.c_int64, C.POINTER(C.c_int64), dp, C.POINTER(C.c_int64)]
        L.dt_threshold_noalloc.argtypes = [vp, vp, vp, C.c_int64, C.c_double, C.c_int32, C.c_int64, vp, vp, vp]
        L.dt_partials_sparse.argtypes = [vp, C.c_int64, vp, vp, vp, vp, C.c_int32, C.POINTER(C.c_int64)]
        L.dt_partials_reset.argtypes = [vp]
        L.dt_partials_add.argtypes = [vp, vp, vp, vp, vp, C.c_int64, C.c_int32]
        L.dt_partials_finalize.argtypes = [vp, vp, vp, C.c_int32]
        L.dt_topk.argtypes = [vp, C.c_int32, C.c_int32, C.POINTER(C.c_int64), dp, ip]
        L.dt_project.argtypes = [vp, dp, C.c_int64, C.c_double, dp, dp, ip]
        L.dt_gather_hits.argtypes = [vp, C.c_int64, C.c_int32, C.c_int32, vp, vp, vp, C.c_int64, vp, vp, vp]
        L.dt_filter_intersections.argtypes = [vp, vp, C.c_int64, C.c_double, C.c_int32, C.c_int32, C.c_int32,
                                              C.POINTER(vp), C.POINTER(vp), C.POINTER(vp),
                                              C.POINTER(C.c_int64), C.POINTER(C.c_int64), ip]
        L.dt_sky_order.argtypes = [vp, vp, vp, C.c_int64, C.c_double, vp]
        L.dt_set_option.argtypes = [vp, C.c_char_p, C.c_int64]
        L.dt_get_stats.argtypes = [vp, C.POINTER(dt_stats)]
        L.dt_last_error.argtypes = [vp]
        L.dt_last_error.restype = C.c_char_p
        L.dt_version.restype = C.c_char_p
        L.dt_fp64_peak.argtypes = [C.c_int32, dp]
        L.dt_probe_random_gather.argtypes = [C.c_int32, C.c_int64, C.c_int32, dp]
        for name in EXPORTS:
            getattr(L, name)
        _lib = L
    return _lib


def _check(rc: int, ctx=None):
    if rc != DT_OK:
        msg = lib().dt_last_error(ctx).decode()        # ctx None: the message of the last context-free call
        raise DtError(rc, msg)


def _is_torch(x) -> bool:
    return type(x).__module__.startswith("torch")


def _ptr_kind(x):
    """(address, mem_kind) of a contiguous numpy array or torch tensor."""
    if x is None:
        return None, DT_MEM_HOST
    if _is_torch(x):
        if not x.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if x.is_cuda:
            return x.data_ptr(), DT_MEM_DEVICE
        return x.data_ptr(), (DT_MEM_PINNED if x.is_pinned() else DT_MEM_HOST)
    if not x.flags["C_CONTIGUOUS"]:
        raise ValueError("array must be C-contiguous")
    return x.ctypes.data, DT_MEM_HOST


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


# ---- the C calls, same names ---------------------------------------------------------------------------
def dt_version() -> str:
    return lib().dt_version().decode()


def dt_create(t, obs_ecl, ra0, dec0, width: int, height: int, pixel_scale: float, gm: float = math.nan,
              c: float = math.nan, obliquity: float = math.nan, variance_mode: int = 0, var_scalar=None,
              device: int = 0, stream: Optional[int] = None, hbm_budget_bytes: int = 0, flags: int = 0):
    """-> opaque context handle (ctypes c_void_p).  Metadata arrays are host arrays (copied)."""
    f = lambda a: np.ascontiguousarray(a, dtype=np.float64)  # noqa: E731
    t, obs_ecl, ra0, dec0 = f(t), f(obs_ecl), f(ra0), f(dec0)
    n = t.size
    if obs_ecl.shape != (n, 3) or ra0.shape != (n,) or dec0.shape != (n,):
        raise ValueError("metadata shapes do not match n_exposures")
    vs = f(var_scalar) if var_scalar is not None else None
    if vs is not None and vs.shape != (n,):
        raise ValueError("var_scalar must have n_exposures entries")
    s = dt_survey(C.sizeof(dt_survey), n, width, height, _dp(t), _dp(obs_ecl), _dp(ra0), _dp(dec0),
                  pixel_scale, gm, c, obliquity, variance_mode, _dp(vs) if vs is not None else None,
                  device, C.c_void_p(stream) if stream else None, hbm_budget_bytes, flags)
    ctx = C.c_void_p()
    _check(lib().dt_create(C.byref(s), C.byref(ctx)))
    return ctx


def dt_destroy(ctx) -> None:
    _check(lib().dt_destroy(ctx))


def dt_load_image_batch(ctx, first_exposure: int, flux, var=None) -> None:
    """flux (and var): [count, H, W] float32, numpy / torch CPU (pinned or not) / torch CUDA."""
    pf, kind = _ptr_kind(flux)
    pv, kind_v = _ptr_kind(var)
    if var is not None and kind_v != kind:
        raise ValueError("flux and var must live in the same kind of memory")
    if str(flux.dtype).split(".")[-1] != "float32":
        raise ValueError("images must be float32")
    count = int(flux.shape[0])
    _check(lib().dt_load_image_batch(ctx, first_exposure, count, pf, pv, kind), ctx)


def dt_stack(ctx, elements, t0, out=None):
    """elements [n, 6] float64 (numpy or torch, host or CUDA) -> (snr [n] f64, hits [n] i32) in the
    same kind of container.  `out` = (snr, hits) supplies the output buffers (same memory kind as the
    elements: e.g. pinned torch tensors reused from call to call, so that the device->host copy does not
    go through freshly allocated pageable memory)."""
    n = int(elements.shape[0])
    pe, kind = _ptr_kind(elements)
    if out is not None:
        snr, hits = out
        ps, kind_s = _ptr_kind(snr)
        ph, kind_h = _ptr_kind(hits)
        host = (DT_MEM_HOST, DT_MEM_PINNED)
        if not (kind_s == kind_h == kind or (kind in host and kind_s in host and kind_h in host)):
            raise ValueError("out buffers must live in the same kind of memory as the elements")
        if int(snr.shape[0]) != n or int(hits.shape[0]) != n:
            raise ValueError("out buffers must have n entries")
        if str(snr.dtype).split(".")[-1] != "float64" or str(hits.dtype).split(".")[-1] != "int32":
            raise ValueError("out = (float64 snr, int32 hits)")
        if str(elements.dtype).split(".")[-1] != "float64":
            raise ValueError("elements must be float64")
    elif _is_torch(elements):
        import torch
        if elements.dtype != torch.float64:
            raise ValueError("elements must be float64")
        snr = torch.empty(n, dtype=torch.float64, device=elements.device)
        hits = torch.empty(n, dtype=torch.int32, device=elements.device)
        ps, ph = snr.data_ptr(), hits.data_ptr()
    else:
        if elements.dtype != np.float64:
            raise ValueError("elements must be float64")
        snr, hits = np.empty(n, np.float64), np.empty(n, np.int32)
        ps, ph = snr.ctypes.data, hits.ctypes.data
    if not (hasattr(t0, "shape") and len(t0.shape) > 0):
        _check(lib().dt_stack(ctx, pe, n, float(t0), kind, ps, ph), ctx)
    else:                                # one epoch per orbit: dt_stack_epochs
        pt, kind_t = _ptr_kind(t0)
        host = (DT_MEM_HOST, DT_MEM_PINNED)
        if int(t0.shape[0]) != n or str(t0.dtype).split(".")[-1] != "float64":
            raise ValueError("per-orbit epochs: [n] float64")
        if not (kind_t == kind or (kind in host and kind_t in host)):
            raise ValueError("epochs must live in the same kind of memory as the elements")
        if kind == DT_MEM_PINNED and kind_t != DT_MEM_PINNED:
            kind = DT_MEM_HOST
        _check(lib().dt_stack_epochs(ctx, pe, pt, n, kind, ps, ph), ctx)
    return snr, hits


def dt_set_patch(ctx, k: int, weights=None) -> None:
    w = np.ascontiguousarray(weights, dtype=np.float64).reshape(-1) if weights is not None else None
    if w is not None and w.size != k * k:
        raise ValueError("weights must have k*k entries")
    _check(lib().dt_set_patch(ctx, k, _dp(w) if w is not None else None), ctx)


def dt_set_outlier_clip(ctx, clip: float) -> None:
    _check(lib().dt_set_outlier_clip(ctx, float(clip)), ctx)


def dt_threshold(ctx, snr_min: float, min_hits: int = 0, max_out: int = 1 << 20):
    """-> (index [m] int64, snr [m] f64, n_found): orbits with SNR >= snr_min, ascending index."""
    idx, val, nf = np.empty(max(max_out, 1), np.int64), np.empty(max(max_out, 1), np.float64), C.c_int64(0)
    _check(lib().dt_threshold(ctx, float(snr_min), min_hits, max_out, idx.ctypes.data_as(C.POINTER(C.c_int64)),
                              _dp(val), C.byref(nf)), ctx)
    m = min(nf.value, max_out)
    return idx[:m].copy(), val[:m].copy(), nf.value


def dt_threshold_noalloc(snr, hits, snr_min: float, min_hits, index_out, snr_out, n_found, stream=None):
    """dt_threshold over DEVICE tensors without any allocation (dtrack.h): snr [n] f64, hits [n] i32 in;
    index_out [max_out] i64, snr_out [max_out] f64 or None, n_found [1] i64 out -- all torch CUDA tensors the
    caller made, on the current device.  Enqueues on `stream` (a torch.cuda.Stream; default: the current one)
    and returns without synchronising.  n <= DT_NOALLOC_MAX_ORBITS, else DtError(DT_ERR_TOO_LARGE)."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(snr.device)
    assert snr.dtype == torch.float64 and hits.dtype == torch.int32 and index_out.dtype == torch.int64
    assert n_found.dtype == torch.int64 and (snr_out is None or snr_out.dtype == torch.float64)
    assert snr.is_contiguous() and hits.is_contiguous() and index_out.is_contiguous() and hits.numel() == snr.numel()
    max_out = index_out.numel() if snr_out is None else min(index_out.numel(), snr_out.numel())
    _check(lib().dt_threshold_noalloc(st.cuda_stream, snr.data_ptr(), hits.data_ptr(), snr.numel(), float(snr_min),
                                      int(min_hits), max_out, index_out.data_ptr(),
                                      snr_out.data_ptr() if snr_out is not None else None, n_found.data_ptr()))


def dt_sky_order(ctx, elements, t0=0.0):
    """elements: torch CUDA tensor [n, 6] f64 (one unit, n <= 2^20) -> torch int64 tensor [n]: the order dt_stack
    processes the unit in (elements[perm] is what its kernels see).  t0: scalar, or a CUDA tensor [n] of epochs."""
    import torch
    n = int(elements.shape[0])
    perm = torch.empty(n, dtype=torch.int32, device=elements.device)
    per_orbit = hasattr(t0, "shape") and len(t0.shape) > 0
    _check(lib().dt_sky_order(ctx, elements.data_ptr(), t0.data_ptr() if per_orbit else None, n,
                              0.0 if per_orbit else float(t0), perm.data_ptr()), ctx)
    return perm.to(torch.int64)


def dt_partials_sparse(ctx, n: int, device=None):
    """The orbits the context's exposure slice has hits for -> (index int64, S f64, Wt f64, hits i32), index
    ascending; torch CUDA tensors when `device` is given, else numpy arrays."""
    nf = C.c_int64(0)
    _check(lib().dt_partials_sparse(ctx, 0, None, None, None, None, DT_MEM_HOST, C.byref(nf)), ctx)      # count only
    m = nf.value
    if device is not None:
        import torch
        idx = torch.empty(m, dtype=torch.int64, device=device)
        S = torch.empty(m, dtype=torch.float64, device=device)
        Wt = torch.empty(m, dtype=torch.float64, device=device)
        h = torch.empty(m, dtype=torch.int32, device=device)
        if m:
            _check(lib().dt_partials_sparse(ctx, m, idx.data_ptr(), S.data_ptr(), Wt.data_ptr(), h.data_ptr(),
                                            DT_MEM_DEVICE, C.byref(nf)), ctx)
        return idx, S, Wt, h
    idx, S, Wt, h = np.empty(m, np.int64), np.empty(m), np.empty(m), np.empty(m, np.int32)
    if m:
        _check(lib().dt_partials_sparse(ctx, m, idx.ctypes.data, S.ctypes.data, Wt.ctypes.data, h.ctypes.data,
                                        DT_MEM_HOST, C.byref(nf)), ctx)
    return idx, S, Wt, h


def dt_partials_reset(ctx) -> None:
    _check(lib().dt_partials_reset(ctx), ctx)


def dt_partials_add(ctx, index, S, Wt, hits) -> None:
    m = int(index.shape[0])
    if m == 0:
        return
    pi, kind = _ptr_kind(index)
    ps, k2 = _ptr_kind(S)
    pw, k3 = _ptr_kind(Wt)
    ph, k4 = _ptr_kind(hits)
    host = (DT_MEM_HOST, DT_MEM_PINNED)
    if not (kind == k2 == k3 == k4 or all(k in host for k in (kind, k2, k3, k4))):
        raise ValueError("a partial-sum list must live in one kind of memory")
    for x, want in ((index, "int64"), (S, "float64"), (Wt, "float64"), (hits, "int32")):
        if str(x.dtype).split(".")[-1] != want or int(x.shape[0]) != m:
            raise ValueError("partial-sum list: (int64 index, float64 S, float64 Wt, int32 hits) of equal length")
    _check(lib().dt_partials_add(ctx, pi, ps, pw, ph, m, DT_MEM_DEVICE if kind == DT_MEM_DEVICE else DT_MEM_HOST), ctx)


def dt_partials_finalize(ctx, n: int, device=None):
    if device is not None:
        import torch
        snr = torch.empty(n, dtype=torch.float64, device=device)
        hits = torch.empty(n, dtype=torch.int32, device=device)
        _check(lib().dt_partials_finalize(ctx, snr.data_ptr(), hits.data_ptr(), DT_MEM_DEVICE), ctx)
        return snr, hits
    snr, hits = np.empty(n, np.float64), np.empty(n, np.int32)
    _check(lib().dt_partials_finalize(ctx, snr.ctypes.data, hits.ctypes.data, DT_MEM_HOST), ctx)
    return snr, hits


def dt_topk(ctx, k: int, min_hits: int = 0):
    idx, val, nf = np.empty(max(k, 1), np.int64), np.empty(max(k, 1), np.float64), C.c_int32(0)
    _check(lib().dt_topk(ctx, k, min_hits, idx.ctypes.data_as(C.POINTER(C.c_int64)), _dp(val), C.byref(nf)),
           ctx)
    return idx[:nf.value].copy(), val[:nf.value].copy()


def dt_project(ctx, elements, t0: float, n_exposures: int):
    """Debug/parity: -> dict(radec [n,N,2], xy [n,N,2], pix [n,N,2] int32) as numpy arrays."""
    el = np.ascontiguousarray(elements, dtype=np.float64).reshape(-1, 6)
    n, N = el.shape[0], n_exposures
    radec, xy = np.empty((n, N, 2)), np.empty((n, N, 2))
    pix = np.empty((n, N, 2), np.int32)
    _check(lib().dt_project(ctx, _dp(el), n, float(t0), _dp(radec), _dp(xy),
                            pix.ctypes.data_as(C.POINTER(C.c_int32))), ctx)
    return dict(radec=radec, xy=xy, pix=pix)


def dt_gather_hits(ctx, n: int, first_exposure: int, n_groups: int, mask, base, offsets, n_hits: int, S, Wt,
                   cnt) -> None:
    """Kernel 3 on a caller-built hit list; all arguments are torch CUDA tensors (see dtrack.h)."""
    for x in (mask, base, offsets, S, Wt, cnt):
        if not (_is_torch(x) and x.is_cuda and x.is_contiguous()):
            raise ValueError("dt_gather_hits takes contiguous CUDA tensors")
    _check(lib().dt_gather_hits(ctx, n, first_exposure, n_groups, mask.data_ptr(), base.data_ptr(),
                                offsets.data_ptr(), n_hits, S.data_ptr(), Wt.data_ptr(), cnt.data_ptr()), ctx)


def dt_filter_intersections(ctx, elements, t0: float, first_exposure: int, n_exposures: int) -> dict:
    """Kernel 1 (+2) for one work unit -> dict(mask, base, offsets: device addresses owned by the context,
    n_hits, n_pad, n_groups); see dtrack.h."""
    pe, kind = _ptr_kind(elements)
    m, b, o = C.c_void_p(), C.c_void_p(), C.c_void_p()
    nh, npad, ng = C.c_int64(), C.c_int64(), C.c_int32()
    _check(lib().dt_filter_intersections(ctx, pe, int(elements.shape[0]), float(t0), kind, first_exposure,
                                         n_exposures, C.byref(m), C.byref(b), C.byref(o), C.byref(nh),
                                         C.byref(npad), C.byref(ng)), ctx)
    return dict(mask=m.value, base=b.value, offsets=o.value, n_hits=nh.value, n_pad=npad.value,
                n_groups=ng.value)


def dt_set_option(ctx, name: str, value: int) -> None:
    _check(lib().dt_set_option(ctx, name.encode(), int(value)), ctx)


def dt_get_stats(ctx) -> dict:
    st = dt_stats()
    st.struct_size = C.sizeof(dt_stats)
    _check(lib().dt_get_stats(ctx, C.byref(st)), ctx)
    return {name: getattr(st, name) for name, _ in dt_stats._fields_ if name != "struct_size"}


def dt_fp64_peak(device: int = 0) -> float:
    out = C.c_double(0.0)
    _check(lib().dt_fp64_peak(device, C.byref(out)))
    return out.value


def dt_probe_random_gather(device: int = 0, buffer_bytes: int = 8 << 30, hint64: int = 0) -> float:
    out = C.c_double(0.0)
    _check(lib().dt_probe_random_gather(device, buffer_bytes, hint64, C.byref(out)))
    return out.value


# ---- convenience wrapper -------------------------------------------------------------------------------
class Tracker:
    """One dt_context.  `Tracker.from_scene(scene)` takes a dtsynth Scene (metadata only)."""

    def __init__(self, t, obs_ecl, ra0, dec0, width, height, pixel_scale, **kw):
        self.n_exposures = int(np.asarray(t).size)
        self.width, self.height = int(width), int(height)
        self.ctx = dt_create(t, obs_ecl, ra0, dec0, width, height, pixel_scale, **kw)

    @classmethod
    def from_scene(cls, scene, **kw):
        kw.setdefault("variance_mode", scene.cfg.variance_mode)
        kw.setdefault("var_scalar", scene.var_scalar)
        return cls(scene.t, scene.obs_ecl, scene.ra0, scene.dec0, scene.cfg.width, scene.cfg.height,
                   scene.pixel_scale, gm=scene.gm, c=scene.c, obliquity=scene.obliquity, **kw)

    def load_image_batch(self, first_exposure, flux, var=None):
        dt_load_image_batch(self.ctx, first_exposure, flux, var)

    def stack(self, elements, t0=0.0, out=None):
        return dt_stack(self.ctx, elements, t0, out)

    def set_patch(self, k, weights=None):
        dt_set_patch(self.ctx, k, weights)

    def set_outlier_clip(self, clip):
        dt_set_outlier_clip(self.ctx, clip)

    def threshold(self, snr_min, min_hits=0, max_out=1 << 20):
        return dt_threshold(self.ctx, snr_min, min_hits, max_out)

    def topk(self, k, min_hits=0):
        return dt_topk(self.ctx, k, min_hits)

    def project(self, elements, t0=0.0):
        return dt_project(self.ctx, elements, t0, self.n_exposures)

    def gather_hits(self, n, first_exposure, n_groups, mask, base, offsets, n_hits, S, Wt, cnt):
        dt_gather_hits(self.ctx, n, first_exposure, n_groups, mask, base, offsets, n_hits, S, Wt, cnt)

    def filter_intersections(self, elements, t0=0.0, first_exposure=0, n_exposures=None):
        ne = min(self.n_exposures - first_exposure, 512) if n_exposures is None else n_exposures
        return dt_filter_intersections(self.ctx, elements, t0, first_exposure, ne)

    def sky_order(self, elements, t0=0.0):
        return dt_sky_order(self.ctx, elements, t0)

    def set_option(self, name, value):
        dt_set_option(self.ctx, name, value)

    def stats(self):
        return dt_get_stats(self.ctx)

    def close(self):
        if self.ctx is not None:
            dt_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
