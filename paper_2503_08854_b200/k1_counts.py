"""FP64-pipe instruction counts of kernel 1 per workload, tied to the kernel sources by hash.

bench.py's roofline of `k_propagate` is "FP64-pipe instructions issued per pair x pairs / time" against
the measured DFMA rate.  The per-pair count depends on the binary AND on the workload's mix of Kepler paths
(cull-quality step, wide step, sub-steps, cold solve, refinement), so it is MEASURED, per workload, with

    ncu --metrics smsp__inst_executed_pipe_fp64.sum,smsp__inst_executed.sum,gpu__time_duration.sum \
        --clock-control none --profile-from-start off -k regex:k_propagate --csv \
        --log-file gpurun_out/k1_<workload>.csv python bench.py --count-k1 <workload>

(`--count-k1` runs kernel 1 over all exposures of the workload at a reduced orbit count -- same seeded distributions,
so the same mix -- twice: an unprofiled pass in which the device-side choice of the kernel-1 variant settles, then the
counted pass after cudaProfilerStart; both variants of a unit are launched and the one not chosen returns at once, so
the sums hold what really ran; the pair count goes to gpurun_out/k1_<workload>.txt) and stored by

    python -m paper_2503_08854_b200.k1_counts gpurun_out/k1_*.csv

in k1_fp64_counts.json next to this file, together with the sha256 of the kernel sources.  bench.py uses a
count only while that hash matches the sources the library was built from; otherwise it reports
`frac: null` ("stale counts") instead of a silently wrong fraction.
"""
from __future__ import annotations

import csv
import hashlib
import json
import os
import re
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
TABLE = os.path.join(HERE, "k1_fp64_counts.json")
KERNEL_SOURCES = ["dt_propagate.cu", "dt_orbit.cuh", "dt_k1.cuh", "dt_tma.cuh"]


def source_hash() -> str:
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(HERE, "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def load() -> dict:
    """-> {"valid": bool, "workloads": {name: {...}}, "why": str}"""
    try:
        with open(TABLE) as f:
            t = json.load(f)
    except Exception as e:                                   # no table: no count, never a guess
        return {"valid": False, "workloads": {}, "why": "no count table (%s)" % e}
    if t.get("source_sha256") != source_hash():
        return {"valid": False, "workloads": t.get("workloads", {}),
                "why": "stale counts: kernel sources changed since the ncu measurement"}
    return {"valid": True, "workloads": t["workloads"], "why": "ncu smsp__inst_executed_pipe_fp64.sum per pair"}


def parse_csv(path: str) -> dict:
    """One `--count-k1` run under ncu -> per-pair counts summed over its k_propagate launches."""
    pairs = None
    workload = None
    sums = {}
    launches = 0
    with open(path) as f:
        lines = f.readlines()
    side = os.path.splitext(path)[0] + ".txt"               # written by bench.py --count-k1 itself
    side_lines = open(side).readlines() if os.path.exists(side) else []
    for ln in lines + side_lines:
        m = re.search(r"COUNT_K1 workload=(\S+) pairs=(\d+) flags=(\d+)", ln)
        if m:
            workload, pairs, flags = m.group(1), int(m.group(2)), int(m.group(3))
    rows = [r for r in csv.reader(l for l in lines if l.startswith('"'))]
    if not rows:
        raise ValueError("%s: no ncu rows" % path)
    hdr = rows[0]
    ik, im, iv = hdr.index("Kernel Name"), hdr.index("Metric Name"), hdr.index("Metric Value")
    iid = hdr.index("ID")
    seen = set()
    for r in rows[1:]:
        if len(r) != len(hdr) or "k_propagate" not in r[ik]:
            continue
        seen.add(r[iid])
        sums[r[im]] = sums.get(r[im], 0.0) + float(r[iv].replace(",", ""))
    launches = len(seen)
    if pairs is None:
        raise ValueError("%s: the COUNT_K1 line of bench.py --count-k1 is missing (log the program's stdout into the "
                         "same file, or pass pairs by hand)" % path)
    return {"workload": workload, "flags": flags, "pairs": pairs, "launches": launches,
            "fp64_per_pair": sums["smsp__inst_executed_pipe_fp64.sum"] * 32.0 / pairs,
            "inst_per_pair": sums["smsp__inst_executed.sum"] * 32.0 / pairs,
            "ncu_time_ms": sums.get("gpu__time_duration.sum", 0.0) * 1e-6}


def main(argv):
    table = {"source_sha256": source_hash(), "kernel_sources": KERNEL_SOURCES,
             "metric": "smsp__inst_executed_pipe_fp64.sum x 32 / pairs (thread-level FP64-pipe instructions per pair)",
             "workloads": {}}
    for path in argv:
        rec = parse_csv(path)
        key = rec.pop("workload") + ("" if rec["flags"] == 0 else "@flags=%d" % rec["flags"])
        table["workloads"][key] = rec
        print(key, rec)
    with open(TABLE, "w") as f:
        json.dump(table, f, indent=1, sort_keys=True)
    print("wrote", TABLE)


if __name__ == "__main__":
    main(sys.argv[1:])
