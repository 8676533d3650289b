#!/usr/bin/env python
"""bench.py -- orbit-exposure pairs/s through propagate + project + cull + gather + stack on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload small_mba[+focused]] [--impl reference]

A step is one pass of the whole hot path (dt_stack: kernels 1-3 + finalisation) over the workload's
candidate orbits against all of its exposures.  The default workload is BASELINE.json configs[1]
("Small MBA": 500 exposures of 2048x2048 fp32, 1e6 orbits), literal/diffuse variant; images are
registered once before the timed region (Algorithm 1: LoadImages once, then batches of orbits).
Prints ONE JSON line.  N > 1: replicas only -- every rank holds the
images and processes its own block of 1e6 seeded orbits (weak scaling, no data-path collective).
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
# FP64-pipe instructions kernel 1 issues per pair on its two paths,
# measured with ncu smsp__inst_executed_pipe_fp64.sum on configs[1] (profiles/r1c_final.md): 50.0 per
# pair with the pre-cull (0.01 % of the pairs refined: cull-quality order-2 warm Kepler step without
# polish or refresh, reciprocal from the MUFU seed, geometric position, cone test) and 130.0 per pair with DT_FLAG_NO_PRECULL (every pair solved
# to full precision and refined; that mode has no cone test, ~6 instructions).  A refined pair
# therefore costs at least 130 + 6 - 50.0 = 86.0 more.  Other workloads take longer Kepler paths (wide
# steps on NEO), so the model under-counts their work: their `frac` is a lower bound.
FP64_SLOTS_COARSE = 50.0     # every pair
FP64_SLOTS_REFINE = 86.0     # refined pairs only, on top
# dram__bytes_read.sum + dram__bytes_write.sum of one k_propagate<3> launch on configs[1], from the
# `ncu --set full` capture summarised in profiles/r1c_final.md (48.35 MB + 19.71 MB)
K1_TRAFFIC_BYTES_SMALL_MBA = 68.05e6


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="small_mba")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--orbits", type=int, default=0, help="override the number of candidate orbits")
    ap.add_argument("--exposures", type=int, default=0, help="override the number of exposures")
    ap.add_argument("--flags", type=int, default=0, help="dt_survey.flags (2: cold Kepler, 4: no pre-cull)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-gather-bench", action="store_true")
    ap.add_argument("--gather-only", action="store_true", help="run only the kernel-3 micro-benchmarks")
    ap.add_argument("--gather-reps", type=int, default=5, help="timed repetitions per kernel-3 regime")
    ap.add_argument("--gather-regimes", default="", help="comma-separated subset of the kernel-3 regimes")
    return ap.parse_args()


def make_config(args):
    name = args.workload
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
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_sample_rate(cfg, n_orb, n_exp_s)
    dt_s = (time.perf_counter() - t0) / max(args.steps, 1)
    value = n_orb * n_exp_s / dt_s
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


def gather_bench(dt, trk, cfg, dev, hbm_gbs, reps=5, regimes=None):
    import torch
    from dtsynth import hitlists
    n = min(cfg.n_orbits, 1 << 20)
    G = max(1, min(cfg.n_exp // 32, 15))
    out = []
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    for name, cluster, density in (regimes or GATHER_REGIMES):
        hl = hitlists.build(n, G, cfg.width, cfg.height, cluster, density, 7, dev)
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
        planes = 2 if cfg.variance_mode == 1 else 1
        bytes_min = (hl["hits"] * 4 + hl["mask"].numel() * 4 + hl["base"].numel() * 8 +
                     hl["unique_sectors"] * 32 * planes + hl["touched_orbits"] * 20)
        gbs = bytes_min / (ms * 1e-3) * 1e-9
        # second bound: a fully divergent 4-B gather is served by the L1 at one lane per clock and SM
        # (measured: the reuse regime, whose pixels hit L1, runs at 0.99 of it)
        props = torch.cuda.get_device_properties(dev)
        l1_rate = props.multi_processor_count * sm_clock_hz(dev.index or 0)
        out.append({"regime": name, "hits": hl["hits"], "unique_sectors": hl["unique_sectors"],
                    "bytes_min": int(bytes_min), "ms": ms, "hits_per_s": hl["hits"] / (ms * 1e-3),
                    "achieved": gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": gbs / hbm_gbs,
                    "l1_gather_bound": {"peak": l1_rate, "unit": "gathers/s",
                                        "frac": hl["hits"] / (ms * 1e-3) / l1_rate}})
        del hl, S, Wt, cnt
        torch.cuda.empty_cache()
    return out


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
def rank_elements(cfg, rank: int, world: int) -> np.ndarray:
    """Rank r of N processes its own block of seeded candidates: indices [r n, (r+1) n) of the
    config's orbit stream (weak scaling; no rank ever needs another rank's orbits or results)."""
    n = cfg.n_orbits
    return ds.elements(cfg, rank * n, (rank + 1) * n) if world > 1 else ds.elements(cfg, 0, n)


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


# ---- B200 arm ----------------------------------------------------------------------------------------------
def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    cfg = make_config(args)
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    import torch
    import torch.distributed as dist
    import paper_2503_08854_b200 as dt                # raises if the CUDA library is unavailable

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # ---- synthetic inputs ----
    trk_holder = {}

    def project_fn(scene, elements, t0):            # scene building uses the LIBRARY's dt_project
        with dt.Tracker.from_scene(scene, device=local_rank) as tmp:
            out = tmp.project(elements, t0)
        return out["radec"], out["pix"]

    scene = ds.build_scene(cfg, project_fn)
    n = cfg.n_orbits
    el_np = rank_elements(cfg, rank, world)
    free_b, _total_b = torch.cuda.mem_get_info()
    beyond_hbm = cfg.image_bytes() > 0.75 * free_b          # the library's own default budget
    kw = {} if beyond_hbm else {"hbm_budget_bytes": cfg.image_bytes() + (1 << 30)}
    trk = dt.Tracker.from_scene(scene, device=local_rank, flags=args.flags, **kw)
    trk_holder["t"] = trk
    keep_alive = []
    if beyond_hbm:
        # the survey does not fit HBM (configs[2]): page-locked host planes, streamed or gathered in place
        # by the library.  The host holds a pool of distinct seeded exposures and exposure j registers
        # pool[j mod POOL] (SURVEY.md 8(d) "Host memory"); pooled planes carry no injected sources.
        POOL = 64
        fpool = torch.empty((POOL, cfg.height, cfg.width), dtype=torch.float32).pin_memory()
        vpool = torch.empty((POOL, cfg.height, cfg.width), dtype=torch.float32).pin_memory() \
            if cfg.variance_mode == 1 else None
        for q in range(POOL):
            fpool[q].copy_(ds.noise_plane_t(cfg, q, dev))
            if vpool is not None:
                vpool[q].fill_(float(scene.var_scalar[q]))
        for j in range(cfg.n_exp):
            q = j % POOL
            trk.load_image_batch(j, fpool[q:q + 1], vpool[q:q + 1] if vpool is not None else None)
        keep_alive = [fpool, vpool]
    else:
        for j in range(cfg.n_exp):
            f = scene.flux_plane_t(j, dev).unsqueeze(0).contiguous()
            v = None
            if cfg.variance_mode == 1:
                v = torch.full((1, cfg.height, cfg.width), float(scene.var_scalar[j]), dtype=torch.float32,
                               device=dev)
            trk.load_image_batch(j, f, v)
    el_dev = torch.from_numpy(el_np).to(dev)
    el_pin = torch.from_numpy(el_np).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.gather_only:
        hbm, src = measured_hbm_peak()
        print(json.dumps({"gather_roofline": {"bound": "hbm", "kernel": "k_gather_dense / k_gather_sparse", "peak_source": src,
                                              "regimes": gather_bench(dt, trk, cfg, dev, hbm, args.gather_reps,
                                                                      pick_regimes(args))}}))
        trk.close()
        return

    # ---- warm-up ----
    for _ in range(max(args.warmup, 3)):
        trk.stack(el_dev, scene.t0)
    barrier()

    # ---- timed region: K steps, device-resident inputs ----
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ms_steps, ms_prop, ms_gath = [], [], []
    stats = None
    wall0 = time.perf_counter()
    for _ in range(args.steps):
        flush.fill_(1)                                 # L2 flush between timed iterations (untimed)
        torch.cuda.synchronize()
        trk.stack(el_dev, scene.t0)                    # synchronises; times itself with CUDA events
        stats = trk.stats()
        ms_steps.append(stats["ms_total"])
        ms_prop.append(stats["ms_propagate"])
        ms_gath.append(stats["ms_gather"])
    barrier()
    wall = time.perf_counter() - wall0
    ms_step = float(np.mean(ms_steps))

    # ---- end to end: host (pinned) elements in, host results out, copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        out_pin = (torch.empty(n, dtype=torch.float64).pin_memory(), torch.empty(n, dtype=torch.int32).pin_memory())
        for _ in range(2):
            trk.stack(el_pin, scene.t0, out=out_pin)
        barrier()
        ms_e2e = []
        for _ in range(args.steps):
            flush.fill_(1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            snr_h, hits_h = trk.stack(el_pin, scene.t0, out=out_pin)
            ms_e2e.append((time.perf_counter() - t0) * 1e3)
        barrier()
        ms_e2e = float(np.mean(ms_e2e))
    clocks = sampler.stop() if sampler else None

    # ---- max over ranks ----
    if world > 1:
        ms_step, ms_e2e_max = max_over_ranks([ms_step, ms_e2e if not args.no_e2e else 0.0], world, dev)
        if not args.no_e2e:
            ms_e2e = ms_e2e_max
    pairs_total = float(cfg.pairs) * world
    value = pairs_total / (ms_step * 1e-3)
    if not args.no_e2e:
        e2e = {"value": pairs_total / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(n * 48),
               "d2h_bytes_per_step": int(n * 12), "ms_per_step": ms_e2e,
               "note": "dt_stack with pinned host elements in, pinned host SNR/hits out; images registered before"}

    if rank == 0:
        # ---- roofline of the dominant kernel (kernel 1: FP64 ALU bound) ----
        peak_tf = dt.dt_fp64_peak(local_rank)
        ms_k1 = float(np.mean(ms_prop)) / max(stats["propagate_launches"], 1)
        pairs_per_launch = cfg.pairs / max(stats["propagate_launches"], 1)
        refined_frac = stats["refined_pairs"] / max(stats["pairs"], 1)
        slots = FP64_SLOTS_COARSE + refined_frac * FP64_SLOTS_REFINE
        if args.flags & 4:
            slots = 130.0
        achieved_tf = 2.0 * slots * pairs_per_launch / (ms_k1 * 1e-3) * 1e-12
        roofline = {"bound": "alu", "kernel": "k_propagate", "achieved": achieved_tf, "peak": peak_tf,
                    "unit": "TFLOP/s", "frac": achieved_tf / peak_tf if peak_tf else None,
                    "traffic": K1_TRAFFIC_BYTES_SMALL_MBA if (cfg.name == "small_mba" and not args.orbits and
                                                              not args.exposures and not args.flags) else None,
                    "traffic_unit": "bytes per launch (ncu dram read + write, profiles/r1c_final.md)",
                    "peak_source": "dt_fp64_peak DFMA probe measured in this run (MEASURED_PEAKS.json has no FP64 figure)",
                    "fp64_slots_per_pair": slots, "refined_fraction": refined_frac,
                    "ms_per_launch": ms_k1, "share_of_step": float(np.mean(ms_prop)) / ms_step}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": cfg.name, "n_orbits": n, "n_exposures": cfg.n_exp,
                           "image": "%dx%d fp32" % (cfg.width, cfg.height),
                           "variance_mode": cfg.variance_mode, "flags": args.flags,
                           "parallelism": "replicas x%d" % world, "l2": "flushed between timed steps",
                           "images_resident": not bool(stats["streamed"]),
                           "image_zero_copy": bool(stats["image_zero_copy"]),
                           "h2d_image_bytes_per_step": int(stats["h2d_image_bytes"])},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(stats["launches"]) * args.steps,
                "roofline": roofline,
                "stages_ms": {"propagate": float(np.mean(ms_prop)), "gather": float(np.mean(ms_gath)),
                              "finalize": stats["ms_finalize"]},
                "hits_per_step": int(stats["hits"]), "cold_solves": int(stats["cold_solves"]), "substep_solves": int(stats["substep_solves"]),
                "wall_s_timed_region": wall}
        if not args.no_gather_bench:
            hbm, src = measured_hbm_peak()
            line["gather_roofline"] = {"bound": "hbm", "kernel": "k_gather_dense / k_gather_sparse", "peak_source": src,
                                       "regimes": gather_bench(dt, trk, cfg, dev, hbm, args.gather_reps,
                                                               pick_regimes(args))}
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(cfg)
        print(json.dumps(line))
    trk.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
