"""CPU-side checks of the product: the C-ABI library builds, loads and exports every symbol that
include/dtrack.h declares; struct layouts of the binding match the header; compute calls fail loudly
(no CPU fallback) on a box without a CUDA device; the product never imports the oracle."""
import ast
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    import paper_2503_08854_b200 as dt
    hdr = open(os.path.join(ROOT, "include", "dtrack.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(dt_[a-z0-9_]+)\s*\(", hdr))
    assert {"dt_create", "dt_load_image_batch", "dt_stack", "dt_topk"} <= declared
    L = dt.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(dt.EXPORTS)
    assert "sm_100a" in dt.dt_version()


def test_binding_struct_layout_matches_header():
    """Compile a tiny C program against the header and compare sizeof/offsetof with ctypes."""
    import subprocess
    import tempfile
    import paper_2503_08854_b200 as dt
    src = r'''
#include <stdio.h>
#include <stddef.h>
#include "dtrack.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu\n", sizeof(dt_survey), offsetof(dt_survey, pixel_scale),
         offsetof(dt_survey, var_scalar), offsetof(dt_survey, hbm_budget_bytes), offsetof(dt_survey, flags),
         offsetof(dt_survey, stream));
  printf("%zu %zu %zu %zu\n", sizeof(dt_stats), offsetof(dt_stats, hits), offsetof(dt_stats, ms_total),
         offsetof(dt_stats, gather_launches));
  return 0; }
'''
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "a.c"), "w").write(src)
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), os.path.join(d, "a.c"), "-o",
                        os.path.join(d, "a")], check=True)
        out = subprocess.run([os.path.join(d, "a")], capture_output=True, text=True, check=True).stdout.split()
    S, T = dt.dt_survey, dt.dt_stats
    want = [C.sizeof(S), S.pixel_scale.offset, S.var_scalar.offset, S.hbm_budget_bytes.offset, S.flags.offset,
            S.stream.offset, C.sizeof(T), T.hits.offset, T.ms_total.offset, T.gather_launches.offset]
    assert [int(x) for x in out] == want


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU-only box")
    import paper_2503_08854_b200 as dt
    with pytest.raises(dt.DtError) as e:
        dt.dt_create(np.zeros(2), np.zeros((2, 3)), np.zeros(2), np.zeros(2), 64, 64, 1e-6,
                     var_scalar=np.ones(2))
    assert e.value.code == dt.DT_ERR_CUDA
    with pytest.raises(dt.DtError):
        dt.dt_fp64_peak(0)


def test_invalid_arguments_rejected_before_any_device_work():
    import paper_2503_08854_b200 as dt
    L = dt.lib()
    assert L.dt_create(None, None) == dt.DT_ERR_INVALID_ARG
    ctx = C.c_void_p()
    s = dt.dt_survey()
    s.struct_size = 4            # wrong ABI size
    assert L.dt_create(C.byref(s), C.byref(ctx)) == dt.DT_ERR_INVALID_ARG
    assert L.dt_destroy(None) == dt.DT_ERR_INVALID_ARG
    assert L.dt_stack(None, None, 0, 0.0, 0, None, None) == dt.DT_ERR_INVALID_ARG
    assert L.dt_last_error(None) is not None


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2503_08854_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            path = os.path.join(dirpath, fn)
            if fn.endswith(".py"):
                tree = ast.parse(open(path).read())
                for node in ast.walk(tree):
                    names = []
                    if isinstance(node, ast.Import):
                        names = [a.name for a in node.names]
                    elif isinstance(node, ast.ImportFrom):
                        names = [node.module or ""]
                    assert not any(n.split(".")[0] == "oracle" for n in names), path
            elif fn.endswith((".cu", ".cuh", ".h")):
                text = open(path).read()
                assert "dt_oracle" not in text and "oracle/" not in text.replace("shares\n// nothing with oracle/", ""), path
