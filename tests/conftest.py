import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_collection_modifyitems(config, items):
    """GPU tests fail loudly (not skip) when selected on a box with a GPU but no extension; on a
    CPU-only box they are deselected by `-m "not gpu"` and skipped if somebody runs them anyway."""
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def read_golden(name):
    """tests/golden/<name>: '#' comments, then 'key value' or 'const key value' lines."""
    vals, consts = {}, {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            p = line.split()
            if p[0] == "const":
                consts[p[1]] = float(p[2])
            else:
                vals[p[0]] = float(p[1])
    return vals, consts


PARITY_REPORT = os.path.join(ROOT, "gpurun_out", "parity_report.json")


def parity_record(case, **counts):
    """north_star: pixel mismatches inside the 1e-6 px guard band are "counted and reported".  Every GPU
    parity test leaves its counts here (gpurun_out/parity_report.json: flagged pairs / orbits, in-band
    mismatches, what was compared); bench.py echoes the file as `parity_report` when it is present."""
    import json
    os.makedirs(os.path.dirname(PARITY_REPORT), exist_ok=True)
    try:
        with open(PARITY_REPORT) as f:
            rep = json.load(f)
    except Exception:
        rep = {}
    rep[case] = {k: (v.item() if hasattr(v, "item") else v) for k, v in counts.items()}
    with open(PARITY_REPORT, "w") as f:
        json.dump(rep, f, indent=1, sort_keys=True)
