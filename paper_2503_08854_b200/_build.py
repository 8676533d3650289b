"""In-tree build of the CUDA library (nvcc, sm_100a only).  `python -m paper_2503_08854_b200._build`

The shared object lands next to this file (git-ignored, but it travels to the GPU box with the
snapshot).  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libdtrack.so")
SOURCES = ["dt_api.cu", "dt_propagate.cu", "dt_gather.cu", "dt_gather_dense.cu", "dt_tiles.cu", "dt_topk.cu", "dt_peak.cu", "dt_sort.cu"]
HEADERS = ["dt_common.cuh", "dt_k1.cuh", "dt_orbit.cuh", "dt_gather.cuh", "dt_tma.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--fmad=true",
              "-Xptxas", "-v"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(INCLUDE, "dtrack.h"),
                                                                 os.path.abspath(__file__)]
    return os.path.getmtime(LIB) < max(os.path.getmtime(d) for d in deps)


LIB_BOUNDS = os.path.join(HERE, "libdtrack_bounds.so")


def build(force: bool = False, verbose: bool = False, bounds: bool = False) -> str:
    """bounds=True: the debug build with device-side bounds checks (-DDT_BOUNDS_CHECK) -> libdtrack_bounds.so; load it
    with DTRACK_LIB=<path> (the binding honours it)."""
    if not bounds and not force and not _stale():
        return LIB
    nvcc = _nvcc()
    objs = []
    log = []
    lib = LIB_BOUNDS if bounds else LIB
    for src in SOURCES:
        obj = os.path.join(CSRC, src.replace(".cu", ".bounds.o" if bounds else ".o"))
        cmd = [nvcc] + NVCC_FLAGS + (["-DDT_BOUNDS_CHECK"] if bounds else []) + \
              ["-I", INCLUDE, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        log.append(r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s\n%s" % (src, r.stdout, r.stderr))
        objs.append(obj)
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib] + objs
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
    if not bounds:
        with open(os.path.join(CSRC, "ptxas.log"), "w") as f:
            f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, bounds="--bounds" in sys.argv))
