"""ctypes front-end of the CPU oracle (oracle/dt_oracle.c).

TEST INFRASTRUCTURE, not product code: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports the CUDA package.
The shared object is built with gcc on first use (`build()`), flags fixed here:
  gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared dt_oracle.c -lm
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dt_oracle.c")
_HDR = os.path.join(_HERE, "dt_oracle.h")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    stale = (not os.path.exists(_LIB)) or force or \
        os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if stale:
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Survey(C.Structure):
    _fields_ = [("n_exposures", C.c_int32), ("width", C.c_int32), ("height", C.c_int32),
                ("t", C.POINTER(C.c_double)), ("obs_ecl", C.POINTER(C.c_double)),
                ("ra0", C.POINTER(C.c_double)), ("dec0", C.POINTER(C.c_double)),
                ("pixel_scale", C.c_double), ("gm", C.c_double), ("c", C.c_double),
                ("obliquity", C.c_double), ("variance_mode", C.c_int32),
                ("var_scalar", C.POINTER(C.c_double))]


class _StackOpts(C.Structure):
    _fields_ = [("patch", C.c_int32), ("weights", C.POINTER(C.c_double)), ("clip", C.c_double),
                ("t0_per_orbit", C.POINTER(C.c_double))]


class PairStruct(C.Structure):
    _fields_ = [("M", C.c_double), ("E", C.c_double), ("r", C.c_double * 3), ("tau", C.c_double),
                ("M1", C.c_double), ("E1", C.c_double), ("r1", C.c_double * 3),
                ("q", C.c_double * 3), ("rho", C.c_double), ("ra", C.c_double), ("dec", C.c_double),
                ("D", C.c_double), ("xi", C.c_double), ("eta", C.c_double),
                ("x", C.c_double), ("y", C.c_double), ("ix", C.c_int32), ("iy", C.c_int32),
                ("hit", C.c_int32), ("flag", C.c_int32), ("kepler_iters", C.c_int32),
                ("kepler_resid", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
        L.dto_kepler.argtypes = [C.c_double, C.c_double, dp, ip, dp]
        L.dto_pq.argtypes = [C.c_double] * 3 + [dp, dp]
        L.dto_pq.restype = None
        L.dto_helio.argtypes = [dp, C.c_double, C.c_double, C.c_double, dp, dp, dp]
        L.dto_pair_chain.argtypes = [C.POINTER(_Survey), dp, C.c_double, C.c_int32,
                                     C.POINTER(PairStruct)]
        L.dto_project.argtypes = [C.POINTER(_Survey), dp, C.c_int64, C.c_double, dp, dp, ip,
                                  C.POINTER(C.c_uint8)]
        L.dto_stack.argtypes = [C.POINTER(_Survey), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                dp, C.c_int64, C.c_double, dp, ip, dp, dp, ip]
        L.dto_topk.argtypes = [dp, ip, C.c_int64, C.c_int32, C.c_int32, C.POINTER(C.c_int64), dp, ip]
        L.dto_stack_ex.argtypes = [C.POINTER(_Survey), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), dp, C.c_int64,
                                   C.c_double, C.POINTER(_StackOpts), dp, ip, dp, dp, ip]
        L.dto_threshold.argtypes = [dp, ip, C.c_int64, C.c_double, C.c_int32, C.c_int64, C.POINTER(C.c_int64), dp,
                                    C.POINTER(C.c_int64)]
        L.dto_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


@dataclass
class Survey:
    """Exposure metadata in the oracle's units (AU, days, rad)."""
    t: np.ndarray
    obs_ecl: np.ndarray
    ra0: np.ndarray
    dec0: np.ndarray
    width: int
    height: int
    pixel_scale: float
    gm: float
    c: float
    obliquity: float
    variance_mode: int = 0
    var_scalar: Optional[np.ndarray] = None

    def __post_init__(self):
        f = lambda a: np.ascontiguousarray(a, dtype=np.float64)  # noqa: E731
        self.t, self.obs_ecl, self.ra0, self.dec0 = f(self.t), f(self.obs_ecl), f(self.ra0), f(self.dec0)
        n = self.t.size
        assert self.obs_ecl.shape == (n, 3) and self.ra0.shape == (n,) and self.dec0.shape == (n,)
        self.var_scalar = f(self.var_scalar) if self.var_scalar is not None else np.ones(n)
        self._c = _Survey(n, self.width, self.height, _dp(self.t), _dp(self.obs_ecl), _dp(self.ra0),
                          _dp(self.dec0), self.pixel_scale, self.gm, self.c, self.obliquity,
                          self.variance_mode, _dp(self.var_scalar))

    @property
    def n_exposures(self) -> int:
        return self.t.size

    @classmethod
    def from_scene(cls, scene) -> "Survey":
        return cls(scene.t, scene.obs_ecl, scene.ra0, scene.dec0, scene.cfg.width, scene.cfg.height,
                   scene.pixel_scale, scene.gm, scene.c, scene.obliquity, scene.cfg.variance_mode,
                   scene.var_scalar)


def kepler(e: float, M: float):
    """-> (E, iterations, residual)"""
    E, it, res = C.c_double(), C.c_int32(), C.c_double()
    rc = lib().dto_kepler(e, M, C.byref(E), C.byref(it), C.byref(res))
    if rc != 0:
        raise ValueError("invalid (e, M)")
    return E.value, it.value, res.value


def pq(inc: float, node: float, peri: float):
    P, Q = np.empty(3), np.empty(3)
    lib().dto_pq(inc, node, peri, _dp(P), _dp(Q))
    return P, Q


def helio(el: Sequence[float], gm: float, t: float, t0: float):
    """-> (r[3], M, E): heliocentric ecliptic position at time t."""
    el = np.ascontiguousarray(el, dtype=np.float64)
    r, M, E = np.empty(3), C.c_double(), C.c_double()
    rc = lib().dto_helio(_dp(el), gm, t, t0, _dp(r), C.byref(M), C.byref(E))
    if rc != 0:
        raise ValueError("invalid orbit")
    return r, M.value, E.value


def pair(survey: Survey, el: Sequence[float], t0: float, j: int) -> PairStruct:
    el = np.ascontiguousarray(el, dtype=np.float64)
    out = PairStruct()
    lib().dto_pair_chain(C.byref(survey._c), _dp(el), t0, j, C.byref(out))
    return out


def project(survey: Survey, elements: np.ndarray, t0: float):
    """-> dict(radec [n,N,2], xy [n,N,2], pix [n,N,2] int32, flag [n,N] uint8)"""
    el = np.ascontiguousarray(elements, dtype=np.float64).reshape(-1, 6)
    n, N = el.shape[0], survey.n_exposures
    radec, xy = np.empty((n, N, 2)), np.empty((n, N, 2))
    pix, flag = np.empty((n, N, 2), np.int32), np.empty((n, N), np.uint8)
    lib().dto_project(C.byref(survey._c), _dp(el), n, t0, _dp(radec), _dp(xy),
                      pix.ctypes.data_as(C.POINTER(C.c_int32)),
                      flag.ctypes.data_as(C.POINTER(C.c_uint8)))
    return dict(radec=radec, xy=xy, pix=pix, flag=flag)


def _plane_ptrs(planes, N):
    if planes is None:
        return None, None
    keep = [np.ascontiguousarray(p, dtype=np.float32) for p in planes]
    assert len(keep) == N
    arr = (C.c_void_p * N)(*[p.ctypes.data for p in keep])
    return arr, keep


def stack(survey: Survey, flux, var, elements: np.ndarray, t0: float):
    """flux/var: sequences of N [H,W] fp32 planes (var None in mode 0).
    -> dict(snr, hits, S, Wt, nflag)"""
    el = np.ascontiguousarray(elements, dtype=np.float64).reshape(-1, 6)
    n, N = el.shape[0], survey.n_exposures
    fp, _keep_f = _plane_ptrs(flux, N)
    vp, _keep_v = _plane_ptrs(var, N)
    snr, S, Wt = np.empty(n), np.empty(n), np.empty(n)
    hits, nflag = np.empty(n, np.int32), np.empty(n, np.int32)
    ip = C.POINTER(C.c_int32)
    rc = lib().dto_stack(C.byref(survey._c), fp, vp, _dp(el), n, t0, _dp(snr),
                         hits.ctypes.data_as(ip), _dp(S), _dp(Wt), nflag.ctypes.data_as(ip))
    if rc != 0:
        raise ValueError("dto_stack failed (%d)" % rc)
    return dict(snr=snr, hits=hits, S=S, Wt=Wt, nflag=nflag)


def stack_ex(survey: Survey, flux, var, elements: np.ndarray, t0: float = 0.0, patch: int = 1, weights=None,
             clip: float = float("inf"), t0_per_orbit=None):
    """Extended stack (dt_oracle.h dto_stack_ex): k x k patch with PSF weights, per-intersection outlier
    clip, per-orbit epochs.  -> dict(snr, hits, S, Wt, nflag)"""
    el = np.ascontiguousarray(elements, dtype=np.float64).reshape(-1, 6)
    n, N = el.shape[0], survey.n_exposures
    fp, _keep_f = _plane_ptrs(flux, N)
    vp, _keep_v = _plane_ptrs(var, N)
    w = np.ascontiguousarray(weights, dtype=np.float64).reshape(-1) if weights is not None else None
    if w is not None:
        assert w.size == patch * patch
    te = np.ascontiguousarray(t0_per_orbit, dtype=np.float64) if t0_per_orbit is not None else None
    if te is not None:
        assert te.shape == (n,)
    opts = _StackOpts(patch, _dp(w) if w is not None else None, clip, _dp(te) if te is not None else None)
    snr, S, Wt = np.empty(n), np.empty(n), np.empty(n)
    hits, nflag = np.empty(n, np.int32), np.empty(n, np.int32)
    ip = C.POINTER(C.c_int32)
    rc = lib().dto_stack_ex(C.byref(survey._c), fp, vp, _dp(el), n, t0, C.byref(opts), _dp(snr),
                            hits.ctypes.data_as(ip), _dp(S), _dp(Wt), nflag.ctypes.data_as(ip))
    if rc != 0:
        raise ValueError("dto_stack_ex failed (%d)" % rc)
    return dict(snr=snr, hits=hits, S=S, Wt=Wt, nflag=nflag)


def threshold(snr: np.ndarray, hits: np.ndarray, snr_min: float, min_hits: int = 0, max_out: int = 1 << 20):
    """-> (index, snr, n_found): every orbit with finite snr >= snr_min and hits >= min_hits, index order."""
    snr = np.ascontiguousarray(snr, dtype=np.float64)
    hits = np.ascontiguousarray(hits, dtype=np.int32)
    idx, val, nf = np.empty(max(max_out, 1), np.int64), np.empty(max(max_out, 1)), C.c_int64()
    rc = lib().dto_threshold(_dp(snr), hits.ctypes.data_as(C.POINTER(C.c_int32)), snr.size, snr_min, min_hits,
                             max_out, idx.ctypes.data_as(C.POINTER(C.c_int64)), _dp(val), C.byref(nf))
    if rc != 0:
        raise ValueError("dto_threshold failed (%d)" % rc)
    m = min(nf.value, max_out)
    return idx[:m].copy(), val[:m].copy(), nf.value


def topk(snr: np.ndarray, hits: np.ndarray, k: int, min_hits: int = 0):
    snr = np.ascontiguousarray(snr, dtype=np.float64)
    hits = np.ascontiguousarray(hits, dtype=np.int32)
    idx, val, nf = np.empty(max(k, 1), np.int64), np.empty(max(k, 1)), C.c_int32()
    rc = lib().dto_topk(_dp(snr), hits.ctypes.data_as(C.POINTER(C.c_int32)), snr.size, k, min_hits,
                        idx.ctypes.data_as(C.POINTER(C.c_int64)), _dp(val), C.byref(nf))
    if rc != 0:
        raise ValueError("dto_topk failed (%d)" % rc)
    return idx[:nf.value].copy(), val[:nf.value].copy()


def num_threads() -> int:
    return lib().dto_num_threads()


def scene_project_fn(scene, elements: np.ndarray, t0: float):
    """project_fn for dtsynth.build_scene backed by the oracle."""
    out = project(Survey.from_scene(scene), elements, t0)
    return out["radec"], out["pix"]
