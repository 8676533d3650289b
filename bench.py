#!/usr/bin/env python
"""bench.py -- orbit-exposure pairs/s through propagate + project + cull + gather + stack on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload small_mba[+focused]] [--impl reference]

A step is one pass of the whole hot path (dt_stack: kernels 1-3 + finalisation) over the workload's
candidate orbits against all of its exposures.  The default workload is the LARGEST single-GPU config,
BASELINE.json configs[4] "TNO long-baseline" at full size (1000 exposures of 4096x4096 fp32 flux + variance
= 134 GB resident in HBM, 1e8 orbits = 1e11 pairs per step) in its focused variant (the one that gives the
gather/stack stage work: 1.2e10 hits per step); images are registered once before the timed region
(Algorithm 1: LoadImages once, then batches of orbits).  On a GPU with less free memory than that needs the
workload falls back to configs[1] and says so.  The same JSON line carries `configs`: every BASELINE.json
config, literal and focused, at full size with its own pairs/s, e2e, stage times, hits, GB/s, FP64 TFLOP/s
and combined roofline; `gather_roofline`: kernel 3 alone on the hit lists kernel 1 really produces and on
controlled lists; `cpu_baseline`: the oracle on the host cores.  See DESIGN.md "Measurement".
N > 1: replicas only -- every rank holds the images and processes its own block of seeded orbits (weak
scaling, no data-path collective).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import dtsynth as ds  # noqa: E402

METRIC = "orbit-exposure pairs/sec (propagate+project+gather+stack)"
UNIT = "pairs/s"
DEFAULT_WORKLOAD = "tno+focused"
FALLBACK_WORKLOAD = "small_mba"            # when the GPU cannot hold 134 GB of images (named in config.workload)
ALL_CONFIGS = ["tiny", "tiny+focused", "small_mba", "small_mba+focused", "lsst", "lsst+focused", "neo", "neo+focused",
               "tno", "tno+focused"]
UNIT_ORBITS, UNIT_EXPOSURES = 1 << 20, 512     # one work unit of the library (dtrack.h dt_filter_intersections)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--configs", default="all", help="'all', 'none' or a comma-separated list: the per-config array")
    ap.add_argument("--configs-budget-s", type=float, default=330.0,
                    help="stop adding entries to `configs` after this many seconds (the rest is listed as skipped)")
    ap.add_argument("--count-k1", default="", help="run ONE dt_stack of this workload at a reduced orbit count "
                    "(for the ncu FP64 instruction count; see paper_2503_08854_b200/k1_counts.py) and exit")
    ap.add_argument("--gather-real", default="", help="comma-separated workloads: kernel 3 alone on the hit list kernel 1 "
                    "produces for the first work unit (2^20 orbits x <= 512 exposures) of each, then exit")
    ap.add_argument("--probe-random-gather", action="store_true",
                    help="run the random-gather / fetch-granularity probe (dt_probe_gather) and exit")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--orbits", type=int, default=0, help="override the number of candidate orbits")
    ap.add_argument("--exposures", type=int, default=0, help="override the number of exposures")
    ap.add_argument("--flags", type=int, default=0, help="dt_survey.flags (2: cold Kepler, 4: no pre-cull)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-gather-bench", action="store_true")
    ap.add_argument("--gather-only", action="store_true", help="run only the kernel-3 micro-benchmarks")
    ap.add_argument("--option", action="append", help="dt_set_option name=value on the workload's context (repeatable)")
    ap.add_argument("--gather-slab", type=int, default=-1, help="dt_set_option gather_slab / gather_schedule 0 (experiments)")
    ap.add_argument("--gather-reps", type=int, default=5, help="timed repetitions per kernel-3 regime")
    ap.add_argument("--gather-regimes", default="", help="comma-separated subset of the kernel-3 regimes")
    return ap.parse_args()


def make_config(args, name=None):
    name = name or args.workload
    base = name.split("+")[0]
    cfg = ds.CONFIGS[base]
    kw = {}
    if args.orbits:
        kw["n_orbits"] = args.orbits
    if args.exposures:
        kw["n_exp"] = args.exposures
    if kw:
        cfg = ds.scaled(cfg, **kw)
    if name.endswith("+focused"):
        cfg = ds.focused(cfg)
    return cfg


# ---- clocks ----------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            p = [x.strip() for x in line.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0]))
                mx.append(float(p[1]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if p[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(sm)}


# ---- reference arm / cpu baseline: the oracle, as it stands, on the host cores ----------------------------
def oracle_sample_rate(cfg, n_orb_sample: int, n_exp_sample: int, planes=None, repeats: int = 1):
    """pairs/s of oracle.stack on the first n_orb_sample orbits x first n_exp_sample exposures."""
    import oracle                                   # cpu_baseline / --impl reference leg only
    sub = ds.scaled(cfg, n_exp=n_exp_sample) if n_exp_sample < cfg.n_exp else cfg
    t = ds.exposure_times(cfg)[:n_exp_sample]
    ra0, dec0 = ds.tangent_points(cfg, ds.exposure_times(cfg)) if cfg.tangent_mode in ("opposition", "band") \
        else (np.zeros(cfg.n_exp), np.zeros(cfg.n_exp))
    sv = oracle.Survey(t, ds.observer_ecliptic(t), ra0[:n_exp_sample], dec0[:n_exp_sample], cfg.width,
                       cfg.height, ds.PIXEL_SCALE, ds.GM_SUN, ds.C_AU_PER_DAY, ds.OBLIQUITY,
                       cfg.variance_mode, ds.variance_scalars(cfg)[:n_exp_sample])
    el = ds.elements(cfg, 0, n_orb_sample)
    if planes is None:
        planes = [ds.noise_plane_np(sub, 0)] * n_exp_sample      # values do not change the work done
    var = planes if cfg.variance_mode == 1 else None
    best = 0.0
    for _ in range(repeats):
        t0 = time.perf_counter()
        oracle.stack(sv, planes, var, el, 0.0)
        dt_s = time.perf_counter() - t0
        best = max(best, n_orb_sample * n_exp_sample / dt_s)
    return best, oracle.num_threads()


def cpu_baseline(cfg, target_seconds: float = 12.0):
    n_exp_s = min(cfg.n_exp, 64)
    probe_orb = 2000
    rate, cores = oracle_sample_rate(cfg, probe_orb, n_exp_s)
    n_orb = int(min(cfg.n_orbits, max(probe_orb, rate * target_seconds / n_exp_s)))
    rate, cores = oracle_sample_rate(cfg, n_orb, n_exp_s)
    return {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "oracle.stack on the first %d orbits x first %d exposures of %s (%.3g pairs)" %
                      (n_orb, n_exp_s, cfg.name, n_orb * n_exp_s)}


def run_reference(args, cfg, rank: int):
    if rank != 0:
        return
    n_exp_s = min(cfg.n_exp, 64)
    rate0, cores = oracle_sample_rate(cfg, 2000, n_exp_s)
    # each step ~2 s of CPU work so that steps + warmup stay within minutes
    n_orb = int(min(cfg.n_orbits, max(2000, rate0 * 2.0 / n_exp_s)))
    for _ in range(args.warmup):
        oracle_sample_rate(cfg, n_orb, n_exp_s)
    rates = []
    for _ in range(args.steps):                      # each step: oracle.stack on the sample (input generation untimed)
        rates.append(oracle_sample_rate(cfg, n_orb, n_exp_s)[0])
    value = float(np.mean(rates)) if rates else 0.0
    dt_s = n_orb * n_exp_s / value if value else 0.0
    sample = "oracle.stack, first %d orbits x first %d exposures of %s per step" % (n_orb, n_exp_s, cfg.name)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt_s * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "n_orbits": cfg.n_orbits, "n_exposures": cfg.n_exp,
                       "image": "%dx%d fp32" % (cfg.width, cfg.height), "reference": "CPU oracle (plain C fp64)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---- small helpers -------------------------------------------------------------------------------------------
def sm_clock_hz(index: int) -> float:
    """Maximum SM clock (the benches run unthrottled at it; bench.py reports the sampled clocks too)."""
    try:
        out = subprocess.run(["nvidia-smi", "-i", str(index), "--query-gpu=clocks.max.sm",
                              "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=10).stdout
        return float(out.strip().splitlines()[0]) * 1e6
    except Exception:
        return 1.965e9


def measured_hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s of B200_PROFILING.md (of fallback)"


# ---- replicas (N > 1): the only cross-rank logic of the path --------------------------------------------
def rank_block(cfg, rank: int, world: int):
    """Rank r of N processes its own block of seeded candidates: indices [r n, (r+1) n) of the
    config's orbit stream (weak scaling; no rank ever needs another rank's orbits or results)."""
    n = cfg.n_orbits
    return (rank * n, (rank + 1) * n) if world > 1 else (0, n)


def rank_elements(cfg, rank: int, world: int) -> np.ndarray:
    lo, hi = rank_block(cfg, rank, world)
    return ds.elements(cfg, lo, hi)


def max_over_ranks(values, world: int, device=None):
    """Element-wise MAX over ranks of a short list of timings (the only collective bench.py issues
    besides the barriers)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    tt = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return [float(v) for v in tt]


def elements_device(cfg, lo, hi, dev, chunk=5_000_000):
    import torch
    out = torch.empty((hi - lo, 6), dtype=torch.float64, device=dev)
    for a in range(lo, hi, chunk):
        b = min(hi, a + chunk)
        out[a - lo:b - lo] = torch.from_numpy(ds.elements(cfg, a, b)).to(dev)
    return out


# ---- one workload: scene, tracker with its images registered, candidate orbits on the device ------------
class Workload:
    POOL = 64          # distinct pinned exposures a beyond-HBM survey cycles through (SURVEY.md 8(d) "Host memory")

    def __init__(self, dt, cfg, dev, local_rank, rank, world, flags=0, same_plane=False):
        import torch
        self.dt, self.cfg, self.dev = dt, cfg, dev

        def project_fn(scene, elements, t0):            # scene building uses the LIBRARY's dt_project
            with dt.Tracker.from_scene(scene, device=local_rank) as tmp:
                out = tmp.project(elements, t0)
            return out["radec"], out["pix"]

        free_b, _total = torch.cuda.mem_get_info()
        orbit_bytes = cfg.n_orbits * (48 + 36 + 12) + (6 << 30)      # elements, sums, results, hit buffers
        self.beyond_hbm = cfg.image_bytes() + orbit_bytes > free_b
        # pooled planes cannot carry per-exposure injected sources
        self.scene = ds.build_scene(cfg, project_fn, inject=not (self.beyond_hbm or same_plane))
        kw = {} if self.beyond_hbm else {"hbm_budget_bytes": cfg.image_bytes() + (1 << 30)}
        sc = self.scene
        P = min(self.POOL, cfg.n_exp)
        if self.beyond_hbm:                              # exposure j carries pool[j % P]: the variance follows the plane
            sc.var_scalar = sc.var_scalar[np.arange(cfg.n_exp) % P].copy()
        self.trk = dt.Tracker.from_scene(self.scene, device=local_rank, flags=flags, **kw)
        self.keep_alive = []
        if self.beyond_hbm:
            fpool = torch.empty((P, cfg.height, cfg.width), dtype=torch.float32).pin_memory()
            vpool = torch.empty((P, cfg.height, cfg.width), dtype=torch.float32).pin_memory() \
                if cfg.variance_mode == 1 else None
            for q in range(P):
                fpool[q].copy_(ds.noise_plane_t(cfg, q, dev))
                if vpool is not None:
                    vpool[q].fill_(float(sc.var_scalar[q]))
            for j in range(cfg.n_exp):
                q = j % P
                self.trk.load_image_batch(j, fpool[q:q + 1], vpool[q:q + 1] if vpool is not None else None)
            self.keep_alive = [fpool, vpool]
        elif same_plane:                                 # timing-only stores: every exposure carries the same seeded plane
            f = ds.noise_plane_t(cfg, 0, dev).unsqueeze(0).contiguous()
            v = torch.ones_like(f) if cfg.variance_mode == 1 else None
            for j in range(cfg.n_exp):
                self.trk.load_image_batch(j, f, v)
            del f, v
        else:
            for j in range(cfg.n_exp):
                f = sc.flux_plane_t(j, dev).unsqueeze(0).contiguous()
                v = None
                if cfg.variance_mode == 1:
                    v = torch.full((1, cfg.height, cfg.width), float(sc.var_scalar[j]), dtype=torch.float32, device=dev)
                self.trk.load_image_batch(j, f, v)
            del f, v
        lo, hi = rank_block(cfg, rank, world)
        self.el_dev = elements_device(cfg, lo, hi, dev)
        self.n = hi - lo

    def close(self):
        import torch
        self.trk.close()
        self.el_dev = None
        self.keep_alive = []
        torch.cuda.empty_cache()


def time_steps(w, steps, warmup, flush, barrier):
    """K timed dt_stack calls, device-resident elements; the library times itself with CUDA events on its stream."""
    import torch
    for _ in range(warmup):
        w.trk.stack(w.el_dev, w.scene.t0)
    barrier()
    ms, prop, gath, stats = [], [], [], None
    for _ in range(steps):
        flush.fill_(1)                                 # L2 flush between timed iterations (untimed)
        torch.cuda.synchronize()
        w.trk.stack(w.el_dev, w.scene.t0)              # synchronises
        stats = w.trk.stats()
        ms.append(stats["ms_total"])
        prop.append(stats["ms_propagate"])
        gath.append(stats["ms_gather"])
    barrier()
    return float(np.mean(ms)), float(np.mean(prop)), float(np.mean(gath)), stats


def time_e2e(w, steps, flush, barrier):
    """The same call end to end: pinned host elements in, pinned host SNR / hits out, copies inside the timed region
    (host wall clock around the synchronous call)."""
    import torch
    el_pin = torch.empty((w.n, 6), dtype=torch.float64).pin_memory()
    el_pin.copy_(w.el_dev)
    out_pin = (torch.empty(w.n, dtype=torch.float64).pin_memory(), torch.empty(w.n, dtype=torch.int32).pin_memory())
    w.trk.stack(el_pin, w.scene.t0, out=out_pin)
    barrier()
    ms = []
    for _ in range(steps):
        flush.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        w.trk.stack(el_pin, w.scene.t0, out=out_pin)
        ms.append((time.perf_counter() - t0) * 1e3)
    barrier()
    del el_pin, out_pin
    return float(np.mean(ms))


# ---- the hit list kernel 1 really produces for ONE work unit: statistics and kernel 3 alone on it -----------
class _Raw:
    def __init__(self, ptr, n, typestr):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False), "version": 2}


def unit_hit_list(w, n_unit=UNIT_ORBITS):
    """dt_filter_intersections on the first work unit (<= 2^20 orbits x <= 512 exposures) -> the library's own hit
    list, its size, and -- by a sort-unique over (exposure, pixel offset) on the device -- the unique 32-B sectors
    and 128-B lines it touches (bytes_min of SURVEY.md 8(d) needs the unique sectors)."""
    import torch
    dev, cfg = w.dev, w.cfg
    n = min(w.n, n_unit)
    ne = min(cfg.n_exp, UNIT_EXPOSURES)
    # in the order dt_stack processes the unit in (sky order, csrc/dt_sort.cu): the list kernel 3 really gets
    el_unit = w.el_dev[:n]
    el_unit = el_unit[w.trk.sky_order(el_unit, w.scene.t0)].contiguous()
    hl = w.trk.filter_intersections(el_unit, w.scene.t0, 0, ne)
    G, n_pad = hl["n_groups"], hl["n_pad"]
    words = 2 if cfg.variance_mode == 1 else 1                     # fp32 words per pixel in the resident store
    px_per_sector = 8 // words
    mask = torch.as_tensor(_Raw(hl["mask"], G * n_pad, "<i4"), device=dev).view(G, n_pad)
    base = torch.as_tensor(_Raw(hl["base"], G * (n_pad // 32), "<i8"), device=dev).view(G, n_pad // 32)
    offs = torch.as_tensor(_Raw(hl["offsets"], max(hl["n_hits"], 1), "<i4"), device=dev)
    sectors = lines = hits = 0
    lane_bits = torch.arange(32, device=dev).view(1, 1, 32)
    touched = torch.zeros(n_pad, dtype=torch.bool, device=dev)
    for g in range(G):
        m = mask[g].to(torch.int64) & 0xFFFFFFFF
        touched |= m != 0
        bits = (m.view(-1, 32, 1) >> lane_bits) & 1                # [tile, lane, exposure]
        cnt_b = bits.sum(1)
        pos = base[g].view(-1, 1, 1) + (torch.cumsum(cnt_b, 1) - cnt_b).view(-1, 1, 32) + (torch.cumsum(bits, 1) - bits)
        sel = bits.bool()
        if not bool(sel.any()):
            continue
        e = offs[pos[sel]].to(torch.int64) & 0xFFFFFFFF
        expo = e >> 27                                             # the entry names its exposure (dt_common.cuh)
        assert bool((expo == lane_bits.expand_as(bits)[sel]).all()), "hit entries do not carry their exposure"
        key = (g * 32 + expo) * (cfg.width * cfg.height) + (e & 0x7FFFFFF)
        hits += int(key.numel())
        sectors += int(torch.unique(key // px_per_sector).numel())          # exposure groups are disjoint
        lines += int(torch.unique(key // (4 * px_per_sector)).numel())
        del bits, pos, sel, e, key
    assert hits == hl["n_hits"]
    return dict(hl=hl, n=n, n_exp=ne, hits=hits, sectors=sectors, lines=lines, touched_orbits=int(touched.sum()),
                mask_bytes=G * n_pad * 4, base_bytes=G * (n_pad // 32) * 8)


def gather_on_unit(w, u, hbm_gbs, flush, reps=5):
    """Kernel 3 alone (dt_gather_hits) on the unit's real hit list, L2 flushed before each repetition."""
    import torch
    dev, hl, n = w.dev, u["hl"], u["n"]
    S = torch.zeros(n, dtype=torch.float64, device=dev)
    Wt = torch.zeros_like(S)
    cnt = torch.zeros(n, dtype=torch.int32, device=dev)
    L = w.dt.lib()
    times = []
    for r in range(reps + 2):
        S.zero_(); Wt.zero_(); cnt.zero_()
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        w.dt._check(L.dt_gather_hits(w.trk.ctx, n, 0, hl["n_groups"], hl["mask"], hl["base"], hl["offsets"], u["hits"],
                                     S.data_ptr(), Wt.data_ptr(), cnt.data_ptr()), w.trk.ctx)
        e1.record()
        torch.cuda.synchronize()
        if r >= 2:
            times.append(e0.elapsed_time(e1))
    assert int(cnt.sum().item()) == u["hits"]
    ms = float(np.mean(times))
    bytes_min = u["hits"] * 4 + u["mask_bytes"] + u["base_bytes"] + u["sectors"] * 32 + u["touched_orbits"] * 20
    gbs = bytes_min / (ms * 1e-3) * 1e-9
    return {"regime": "real:" + w.cfg.name, "orbits": n, "exposures": u["n_exp"], "hits": u["hits"],
            "unique_sectors": u["sectors"], "unique_lines": u["lines"], "bytes_min": int(bytes_min), "ms": ms,
            "hits_per_s": u["hits"] / (ms * 1e-3), "achieved": gbs, "peak": hbm_gbs, "unit": "GB/s",
            "frac": gbs / hbm_gbs,
            "line_fetch_bound": {"note": "DRAM bytes if every touched 128-B line is fetched exactly once, at the HBM peak",
                                 "frac": (u["lines"] * 128 + u["hits"] * 4 + u["mask_bytes"]) / (ms * 1e-3) * 1e-9 / hbm_gbs}}


# ---- kernel 3 micro-benchmarks (controlled hit lists over the workload's image set) ------
GATHER_REGIMES = [
    # name, cluster window (px), hit density per pair
    ("L0_uniform_dense", 1 << 30, 1.0),
    ("L0_uniform_sparse", 1 << 30, 0.05),
    ("L1_clustered", 256, 1.0),
    ("L2_reuse", 32, 1.0),
]


def pick_regimes(args):
    if not args.gather_regimes:
        return None
    want = set(args.gather_regimes.split(","))
    return [r for r in GATHER_REGIMES if r[0] in want]


def gather_bench(dt, trk, cfg, dev, hbm_gbs, flush, reps=5, regimes=None):
    import torch
    from dtsynth import hitlists
    n = min(cfg.n_orbits, 1 << 20)
    G = max(1, min(cfg.n_exp // 32, 15))
    out = []
    l2_rate = None
    words = 2 if cfg.variance_mode == 1 else 1
    for name, cluster, density in (regimes or GATHER_REGIMES):
        hl = hitlists.build(n, G, cfg.width, cfg.height, cluster, density, 7, dev, px_per_sector=8 // words)
        S = torch.zeros(n, dtype=torch.float64, device=dev)
        Wt = torch.zeros(n, dtype=torch.float64, device=dev)
        cnt = torch.zeros(n, dtype=torch.int32, device=dev)
        times = []
        for r in range(reps + 2):
            S.zero_(); Wt.zero_(); cnt.zero_()
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            trk.gather_hits(n, 0, G, hl["mask"], hl["base"], hl["offsets"], hl["hits"], S, Wt, cnt)
            e1.record()
            torch.cuda.synchronize()
            if r >= 2:
                times.append(e0.elapsed_time(e1))
        assert int(cnt.sum().item()) == hl["hits"]
        ms = float(np.mean(times))
        bytes_min = (hl["hits"] * 4 + hl["mask"].numel() * 4 + hl["base"].numel() * 8 +
                     hl["unique_sectors"] * 32 + hl["touched_orbits"] * 20)
        gbs = bytes_min / (ms * 1e-3) * 1e-9
        # second bound: a fully divergent 4-B gather is served by the L1 at one lane per clock and SM at best;
        # third: the rate the part really gives fully divergent gathers that HIT the L2 (measured by the probe over
        # one 16 MiB plane-sized buffer): the dense schedule keeps the planes L2-resident, so this is its ceiling
        props = torch.cuda.get_device_properties(dev)
        l1_rate = props.multi_processor_count * sm_clock_hz(dev.index or 0)
        if l2_rate is None:
            l2_rate = dt.dt_probe_random_gather(dev.index or 0, 16 << 20, 0)
        out.append({"regime": name, "image_set": cfg.name, "hits": hl["hits"], "unique_sectors": hl["unique_sectors"],
                    "bytes_min": int(bytes_min), "ms": ms, "hits_per_s": hl["hits"] / (ms * 1e-3),
                    "achieved": gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": gbs / hbm_gbs,
                    "l1_gather_bound": {"peak": l1_rate, "unit": "gathers/s",
                                        "frac": hl["hits"] / (ms * 1e-3) / l1_rate},
                    "l2_gather_bound": {"peak": l2_rate, "unit": "gathers/s",
                                        "peak_source": "dt_probe_random_gather over a 16 MiB (L2-resident) buffer, this run",
                                        "frac": hl["hits"] / (ms * 1e-3) / l2_rate}})
        del hl, S, Wt, cnt
        torch.cuda.empty_cache()
    return out


# ---- rooflines -------------------------------------------------------------------------------------------------
def k1_roofline(name, flags, stats, ms_prop, pairs, peak_tf, counts, issue_peak=None):
    """Kernel 1 (propagate + project + cull + compact): plain ALUs, two ceilings.  (1) The FP64 pipe: `achieved` counts
    every FP64-PIPE instruction the kernel issues (FMA, add, mul, compare, convert alike) as one issue slot = 2 flop,
    i.e. it is the FP64-pipe utilisation expressed in TFLOP/s, against the DFMA rate measured in this run -- what
    bounds the pairs that are refined.  (2) The issue slots: every warp instruction of whatever pipe against
    4 schedulers x 1 instruction per clock x SMs x the SM clock -- what bounds the pairs the FP32 group gate removes.
    `frac` is the FP64 fraction; `issue` holds the second; `binding` names the larger.  The per-pair counts are ncu's
    for THIS workload and binary (paper_2503_08854_b200/k1_counts.py); without a valid count frac is null."""
    launches = max(stats["propagate_launches"], 1)
    key = name + ("" if flags == 0 else "@flags=%d" % flags)
    rec = counts["workloads"].get(key) if counts["valid"] else None
    r = {"bound": "alu", "kernel": "k_propagate", "peak": peak_tf, "unit": "TFLOP/s",
         "peak_source": "dt_fp64_peak DFMA probe measured in this run (MEASURED_PEAKS.json has no FP64 figure)",
         "ms_per_launch": ms_prop / launches, "launches_per_step": launches,
         "refined_fraction": stats["refined_pairs"] / max(stats["pairs"], 1), "traffic": None}
    if rec is None:
        r.update(achieved=None, frac=None, fp64_slots_per_pair=None,
                 note=counts["why"] if not counts["valid"] else "no ncu count for workload %r" % key)
        return r
    slots = rec["fp64_per_pair"]
    achieved = 2.0 * slots * pairs / (ms_prop * 1e-3) * 1e-12
    r.update(achieved=achieved, frac=achieved / peak_tf if peak_tf else None, fp64_slots_per_pair=slots,
             inst_per_pair=rec["inst_per_pair"],
             note="FP64-pipe utilisation: ncu smsp__inst_executed_pipe_fp64 per pair of this workload x pairs / time")
    if issue_peak:
        rate = rec["inst_per_pair"] / 32.0 * pairs / (ms_prop * 1e-3)             # warp instructions per second
        r["issue"] = {"achieved": rate * 1e-9, "peak": issue_peak * 1e-9, "unit": "G warp-instructions/s",
                      "frac": rate / issue_peak,
                      "peak_source": "SMs x 4 schedulers x 1 instruction per clock x max SM clock (B200_PROFILING.md)"}
        r["binding"] = "issue" if r["issue"]["frac"] > (r["frac"] or 0.0) else "fp64"
    return r


def combined_roofline(w, stats, ms_step, ms_prop, u, k1, hbm_gbs, h2d_gbs, peak_tf):
    """north_star: time_roof = max(FP64 slots / FP64 peak, gathered + streamed bytes / HBM bandwidth) (+ host-to-
    device time when image batches are streamed); frac = time_roof / measured time of the step."""
    n, pairs, hits = w.n, float(stats["pairs"]), float(stats["hits"])
    # unique 32-B sectors per hit: counted on the first work unit's list, scaled to the step's hits
    sect_per_hit = (u["sectors"] / u["hits"]) if u and u["hits"] else 1.0
    touched = min(float(n), hits)
    bytes_min = n * 48 + n * 12 + pairs / 8 + hits * 8 + hits * sect_per_hit * 32 + touched * 20
    t_hbm = bytes_min / (hbm_gbs * 1e9)
    t_fp64 = (k1["fp64_slots_per_pair"] * pairs / (peak_tf * 1e12 / 2.0)) if k1.get("fp64_slots_per_pair") else None
    if t_fp64 is not None and k1.get("issue"):            # the ALU roof of kernel 1 is the slower of its two ceilings
        t_fp64 = max(t_fp64, k1["inst_per_pair"] / 32.0 * pairs / (k1["issue"]["peak"] * 1e9))
    t_h2d = stats["h2d_image_bytes"] / (h2d_gbs * 1e9) if h2d_gbs else 0.0
    roof = (max(t_fp64, t_hbm) if t_fp64 is not None else None)
    out = {"bytes_min": bytes_min, "t_hbm_ms": t_hbm * 1e3, "t_fp64_ms": None if t_fp64 is None else t_fp64 * 1e3,
           "t_h2d_ms": t_h2d * 1e3, "bound": None, "time_roof_ms": None, "frac": None,
           "gb_per_s": bytes_min / (ms_step * 1e-3) * 1e-9,
           "sectors_per_hit": sect_per_hit, "sectors_from": "first work unit" if u and u["hits"] else "no hits: 1 assumed"}
    if roof is not None:
        out["bound"] = ("h2d" if t_h2d > roof else ("alu" if t_fp64 >= t_hbm else "hbm"))
        out["time_roof_ms"] = (roof + t_h2d) * 1e3
        out["frac"] = (roof + t_h2d) * 1e3 / ms_step
    return out


def h2d_rate_gbs(dev):
    """Pinned host -> device copy rate (the streaming roofline's denominator), 1 GiB, best of 3."""
    import torch
    src = torch.empty(1 << 30, dtype=torch.uint8).pin_memory()
    dst = torch.empty(1 << 30, dtype=torch.uint8, device=dev)
    best = 0.0
    for _ in range(4):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        dst.copy_(src, non_blocking=True)
        e1.record()
        torch.cuda.synchronize()
        best = max(best, (1 << 30) / (e0.elapsed_time(e1) * 1e-3) * 1e-9)
    return best


def run_config(dt, args, name, dev, local_rank, rank, world, steps, warmup, flush, barrier, peaks, counts,
               with_e2e=True, with_gather=True, sample_clocks=False):
    """One workload at full size -> its entry of `configs` (and the pieces of the headline line)."""
    cfg = make_config(args, name) if name == args.workload else ds.CONFIGS[name.split("+")[0]]
    if name.endswith("+focused") and not cfg.name.endswith("+focused"):
        cfg = ds.focused(cfg)
    t_build = time.perf_counter()
    w = Workload(dt, cfg, dev, local_rank, rank, world, flags=args.flags)
    for kv in (args.option or []):                    # dt_set_option name=value (tuning experiments)
        k, _, v = kv.partition("=")
        w.trk.set_option(k, int(v))
    t_build = time.perf_counter() - t_build
    try:
        sampler = ClockSampler(local_rank) if (sample_clocks and rank == 0) else None     # the timed region only
        wall0 = time.perf_counter()
        ms_step, ms_prop, ms_gath, stats = time_steps(w, steps, warmup, flush, barrier)
        ms_e2e = time_e2e(w, max(1, min(steps, 3)), flush, barrier) if with_e2e else None
        wall = time.perf_counter() - wall0
        clocks = sampler.stop() if sampler else None
        if world > 1:
            ms_step, ms_e2e_m = max_over_ranks([ms_step, ms_e2e or 0.0], world, dev)
            ms_e2e = ms_e2e_m if with_e2e else None
        pairs_rank = float(cfg.n_orbits) * cfg.n_exp
        entry = {"workload": cfg.name, "n_orbits": w.n, "n_exposures": cfg.n_exp,
                 "image": "%dx%d fp32%s" % (cfg.width, cfg.height, " flux+variance" if cfg.variance_mode == 1 else ""),
                 "pairs_per_step": pairs_rank * world, "steps": steps, "ms_per_step": ms_step,
                 "pairs_per_s": pairs_rank * world / (ms_step * 1e-3),
                 "e2e_pairs_per_s": (pairs_rank * world / (ms_e2e * 1e-3)) if ms_e2e else None, "e2e_ms_per_step": ms_e2e,
                 "stages_ms": {"propagate": ms_prop, "gather": ms_gath, "finalize": stats["ms_finalize"]},
                 "hits_per_step": int(stats["hits"]), "refined_pairs": int(stats["refined_pairs"]),
                 "cold_solves": int(stats["cold_solves"]), "substep_solves": int(stats["substep_solves"]),
                 "gated_pairs": int(stats["gated_pairs"]),
                 "launches_per_step": int(stats["launches"]),
                 "images_resident": not bool(stats["streamed"]), "image_zero_copy": bool(stats["image_zero_copy"]),
                 "h2d_image_bytes_per_step": int(stats["h2d_image_bytes"]), "build_s": t_build,
                 "wall_s_timed_region": wall}
        if clocks is not None:
            entry["clocks"] = clocks
        u = None
        if rank == 0:
            import torch
            issue_peak = torch.cuda.get_device_properties(dev).multi_processor_count * 4 * sm_clock_hz(local_rank)
            k1 = k1_roofline(cfg.name, args.flags, stats, ms_prop, pairs_rank, peaks["fp64_tf"], counts, issue_peak)
            entry["fp64_tflops"] = k1["achieved"]
            entry["k1_roofline"] = k1
            if with_gather and stats["hits"] > 0 and not w.beyond_hbm:
                u = unit_hit_list(w)
                if u["hits"] >= (1 << 16):                      # kernel 3 alone on the list kernel 1 produced
                    entry["gather_roofline"] = gather_on_unit(w, u, peaks["hbm_gbs"], flush)
            entry["roofline"] = combined_roofline(w, stats, ms_step, ms_prop, u, k1, peaks["hbm_gbs"], peaks["h2d_gbs"],
                                                  peaks["fp64_tf"])
        return entry, w, stats
    except Exception:
        w.close()
        raise


def parity_report():
    """What the GPU parity tests left behind (tests/conftest.py parity_record): north_star asks that pixel
    mismatches inside the 1e-6 px guard band be counted and reported."""
    path = os.path.join(ROOT, "gpurun_out", "parity_report.json")
    try:
        with open(path) as f:
            rep = json.load(f)
    except Exception:
        return None
    tot = {"cases": len(rep)}
    for key in ("flagged_pairs", "flagged_orbits", "flagged", "in_band_pixel_mismatches", "flagged_hit_mismatch"):
        tot[key] = int(sum(v.get(key, 0) for v in rep.values()))
    return {"source": "gpurun_out/parity_report.json (written by pytest -m gpu)", "totals": tot, "cases": rep}


# ---- B200 arm ----------------------------------------------------------------------------------------------
def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, make_config(args), rank)
        return

    import torch
    import torch.distributed as dist
    import paper_2503_08854_b200 as dt                # raises if the CUDA library is unavailable
    from paper_2503_08854_b200 import k1_counts

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.probe_random_gather:
        out = {}
        for hint in (0, 1):
            out["ld.global.nc" + (".L2::64B" if hint else "")] = dt.dt_probe_random_gather(local_rank, 8 << 30, hint)
        res = dt.dt_probe_random_gather(local_rank, 16 << 20, 0)
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        print(json.dumps({"probe_random_gather": {"unit": "4-B gathers/s over an 8 GiB buffer", **out,
                                                  "l2_resident_16MiB": res,
                                                  "l2_resident_lanes_per_clock_and_sm": res / (sms * sm_clock_hz(local_rank))}}))
        return

    if args.count_k1:
        # ONE dt_stack at a reduced orbit count (same seeded distributions => same mix of Kepler paths): the run
        # `ncu --metrics smsp__inst_executed_pipe_fp64.sum ...` profiles (paper_2503_08854_b200/k1_counts.py)
        name = args.count_k1
        cfg = ds.CONFIGS[name.split("+")[0]]
        cfg = ds.scaled(cfg, n_orbits=min(cfg.n_orbits, args.orbits or UNIT_ORBITS))   # full image size, all exposures
        if name.endswith("+focused"):
            cfg = ds.focused(cfg)

        def project_fn(scene, elements, t0):
            with dt.Tracker.from_scene(scene, device=local_rank) as tmp:
                out = tmp.project(elements, t0)
            return out["radec"], out["pix"]

        scene = ds.build_scene(cfg, project_fn, inject=False)
        el = elements_device(cfg, 0, cfg.n_orbits, dev)
        st = {"pairs": 0, "hits": 0, "propagate_launches": 0}
        with dt.Tracker.from_scene(scene, device=local_rank, flags=args.flags) as trk:      # kernel 1 needs no images
            el = el[trk.sky_order(el, scene.t0)].contiguous()        # the order dt_stack processes the unit in
            # pass 0, unprofiled (the ncu command says --profile-from-start off): the device-side choice of the
            # kernel-1 variant settles, as it has for all but the first of a full step's ~100 units; pass 1 is counted
            for counted in (False, True):
                if counted:
                    torch.cuda.synchronize()
                    torch.cuda.cudart().cudaProfilerStart()
                for first in range(0, cfg.n_exp, UNIT_EXPOSURES):
                    ne = min(UNIT_EXPOSURES, cfg.n_exp - first)
                    hl = trk.filter_intersections(el, scene.t0, first, ne)
                    if counted:
                        st["pairs"] += cfg.n_orbits * ne
                        st["hits"] += hl["n_hits"]
                        st["propagate_launches"] += 1
            torch.cuda.synchronize()
            torch.cuda.cudart().cudaProfilerStop()
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        line = "COUNT_K1 workload=%s pairs=%d flags=%d launches=%d hits=%d" % (
            name, st["pairs"], args.flags, st["propagate_launches"], st["hits"])
        with open(os.path.join(ROOT, "gpurun_out", "k1_%s.txt" % name.replace("+", "_")), "w") as f:
            f.write(line + "\n")
        print(line)
        return

    hbm_gbs, hbm_src = measured_hbm_peak()
    if args.gather_real:
        # kernel 3 alone on real hit lists: one work unit per workload; the image VALUES do not matter to the timing, so
        # one seeded plane is registered for every exposure (resident store of the unit's exposures only)
        regs = []
        for name in args.gather_real.split(","):
            cfg = ds.CONFIGS[name.split("+")[0]]
            cfg = ds.scaled(cfg, n_orbits=min(cfg.n_orbits, UNIT_ORBITS), n_exp=min(cfg.n_exp, UNIT_EXPOSURES))
            if name.endswith("+focused"):
                cfg = ds.focused(cfg)
            w = Workload(dt, cfg, dev, local_rank, 0, 1, flags=args.flags, same_plane=True)
            if args.gather_slab >= 0:
                w.trk.set_option("gather_schedule", 0)
                w.trk.set_option("gather_slab", args.gather_slab)
            u = unit_hit_list(w)
            regs.append(gather_on_unit(w, u, hbm_gbs, flush, args.gather_reps))
            w.close()
        print(json.dumps({"gather_roofline": {"bound": "hbm", "kernel": "k_gather_sparse / k_gather_dense",
                                              "peak_source": hbm_src, "regimes": regs}}))
        return
    if args.gather_only:
        cfg = make_config(args, args.workload if args.workload != DEFAULT_WORKLOAD else "small_mba")
        w = Workload(dt, cfg, dev, local_rank, 0, 1, flags=args.flags)
        regs = gather_bench(dt, w.trk, cfg, dev, hbm_gbs, flush, args.gather_reps, pick_regimes(args))
        print(json.dumps({"gather_roofline": {"bound": "hbm", "kernel": "k_gather_dense / k_gather_sparse",
                                              "peak_source": hbm_src, "regimes": regs}}))
        w.close()
        return

    # ---- peaks measured in this run ----
    peaks = {"hbm_gbs": hbm_gbs, "hbm_source": hbm_src, "fp64_tf": dt.dt_fp64_peak(local_rank),
             "h2d_gbs": h2d_rate_gbs(dev)}
    counts = k1_counts.load()

    # ---- the headline workload: the largest single-GPU config when it fits, else the fallback ----
    name = args.workload
    cfg0 = make_config(args, name)
    free_b, _tot = torch.cuda.mem_get_info()
    fits_hbm = cfg0.image_bytes() + cfg0.n_orbits * 96 + (8 << 30) < free_b
    fallback = None
    if name == DEFAULT_WORKLOAD and not args.orbits and not args.exposures and not fits_hbm:
        fallback = "%s needs %.0f GB of HBM, %.0f GB are free: fell back to %s" % (
            name, (cfg0.image_bytes() + cfg0.n_orbits * 96) / 1e9, free_b / 1e9, FALLBACK_WORKLOAD)
        name = FALLBACK_WORKLOAD
    t_start = time.perf_counter()
    entry, w, stats = run_config(dt, args, name, dev, local_rank, rank, world, args.steps, max(args.warmup, 3), flush,
                                 barrier, peaks, counts, with_e2e=not args.no_e2e, with_gather=not args.no_gather_bench,
                                 sample_clocks=True)
    wall = entry["wall_s_timed_region"]
    clocks = entry.pop("clocks", None)
    main_cfg = w.cfg
    n_main = w.n
    topk_ms = {}
    if rank == 0:                                      # device top-k / threshold over the step's per-orbit SNR
        w.trk.stack(w.el_dev, w.scene.t0)              # (the real-hit-list roofline ran dt_filter_intersections since)
        for k in (64, 4096):
            w.trk.topk(k, min_hits=1)
            t0 = time.perf_counter()
            for _ in range(5):
                w.trk.topk(k, min_hits=1)
            topk_ms["k=%d" % k] = (time.perf_counter() - t0) / 5 * 1e3
        t0 = time.perf_counter()
        _i, _v, nf = w.trk.threshold(5.0, min_hits=1)
        topk_ms["threshold snr>=5"] = (time.perf_counter() - t0) * 1e3
        topk_ms["n_above_5"] = int(nf)
    controlled = []
    if rank == 0 and main_cfg.name == "small_mba" and not args.no_gather_bench:
        controlled = gather_bench(dt, w.trk, w.cfg, dev, hbm_gbs, flush, args.gather_reps, pick_regimes(args))
    w.close()

    line = None
    if rank == 0:
        k1 = entry["k1_roofline"]
        k1["share_of_step"] = entry["stages_ms"]["propagate"] / entry["ms_per_step"]
        line = {"metric": METRIC, "value": entry["pairs_per_s"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": entry["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": entry["workload"], "n_orbits": n_main, "n_exposures": main_cfg.n_exp,
                           "image": entry["image"], "variance_mode": main_cfg.variance_mode, "flags": args.flags,
                           "parallelism": "replicas x%d" % world, "l2": "flushed between timed steps",
                           "images_resident": entry["images_resident"], "image_zero_copy": entry["image_zero_copy"],
                           "h2d_image_bytes_per_step": entry["h2d_image_bytes_per_step"], "fallback": fallback},
                "clocks": clocks,
                "e2e": None if entry["e2e_pairs_per_s"] is None else {
                    "value": entry["e2e_pairs_per_s"], "unit": UNIT, "h2d_bytes_per_step": int(n_main * 48),
                    "d2h_bytes_per_step": int(n_main * 12), "ms_per_step": entry["e2e_ms_per_step"],
                    "note": "dt_stack with pinned host elements in, pinned host SNR/hits out; images registered before"},
                "gpu_launches": entry["launches_per_step"] * args.steps,
                "roofline": k1, "step_roofline": entry.get("roofline"),
                "stages_ms": entry["stages_ms"], "hits_per_step": entry["hits_per_step"],
                "cold_solves": entry["cold_solves"], "substep_solves": entry["substep_solves"],
                "gated_pairs": entry["gated_pairs"],
                "topk_ms": topk_ms, "peaks": peaks, "wall_s_timed_region": wall}

    # ---- every BASELINE.json config, literal and focused, at full size ----
    configs, gather_regimes, skipped = [entry], list(controlled), []
    if "gather_roofline" in entry:
        gather_regimes.append(entry["gather_roofline"])
    want = [] if args.configs == "none" else (ALL_CONFIGS if args.configs == "all" else args.configs.split(","))
    for cname in want:
        if cname == entry["workload"]:
            continue
        if time.perf_counter() - t_start > args.configs_budget_s:
            skipped.append(cname)
            continue
        small = cname.startswith("tiny") or cname.startswith("small_mba")
        try:
            e, wc, _st = run_config(dt, args, cname, dev, local_rank, rank, world, 20 if small else 2, 3 if small else 1,
                                    flush, barrier, peaks, counts, with_e2e=not args.no_e2e,
                                    with_gather=not args.no_gather_bench)
        except Exception as ex:                       # e.g. not enough host memory for the pinned pool
            skipped.append("%s (%s)" % (cname, str(ex)[:120]))
            continue
        if rank == 0 and cname == "small_mba" and not args.no_gather_bench:
            # controlled hit lists over this image set (SURVEY.md 8(d) regimes L0 / L1 / L2)
            gather_regimes += gather_bench(dt, wc.trk, wc.cfg, dev, hbm_gbs, flush, args.gather_reps, pick_regimes(args))
        wc.close()
        if "gather_roofline" in e:
            gather_regimes.append(e["gather_roofline"])
        configs.append(e)

    if rank == 0:
        line["configs"] = configs
        line["configs_skipped"] = skipped
        if gather_regimes:
            line["gather_roofline"] = {"bound": "hbm", "kernel": "k_gather_sparse / k_gather_dense", "peak_source": hbm_src,
                                       "regimes": gather_regimes}
        pr = parity_report()
        if pr:
            line["parity_report"] = pr
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(main_cfg)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
