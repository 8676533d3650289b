"""The seeded input generators (dtsynth/): reproducibility and workload structure.  CPU only."""
import ast
import math
import os

import numpy as np
import torch

import dtsynth as ds
import oracle
from dtsynth import rng


def test_rng_numpy_and_torch_agree_bitwise():
    k = np.arange(0, 200000, dtype=np.int64)
    for seed, stream in [(0, 1), (3, rng.STREAM_NOISE_BASE + 7), (12345, 22)]:
        h_np = rng.hash_np(seed, stream, k)
        h_t = rng.hash_t(seed, stream, torch.from_numpy(k)).numpy().view(np.uint64)
        assert np.array_equal(h_np, h_t)
        u_np = rng.uniform_np(seed, stream, k)
        assert np.array_equal(u_np, rng.uniform_t(seed, stream, torch.from_numpy(k)).numpy())
        assert u_np.min() > 0.0 and u_np.max() < 1.0
    z_np = rng.normal_np(5, 100, 101, k)
    z_t = rng.normal_t(5, 100, 101, torch.from_numpy(k)).numpy()
    assert np.array_equal(z_np, z_t)
    assert np.array_equal(z_np.astype(np.float32).astype(np.float64), z_np)   # fp32-exact
    assert abs(z_np.mean()) < 0.01 and abs(z_np.std() - 1.0) < 0.01


def test_subranges_regenerate():
    cfg = ds.CONFIGS["small_mba"]
    a = ds.elements(cfg, 1000, 1100)
    b = ds.elements(cfg, 0, 2000)[1000:1100]
    assert np.array_equal(a, b)
    assert a[:, 0].min() >= 2.1 and a[:, 0].max() <= 3.3 and a[:, 1].max() <= 0.3
    small = ds.scaled(cfg, width=64, height=64)
    p = ds.noise_plane_np(small, 3)
    assert np.array_equal(ds.noise_values_np(small, 3, np.array([5, 77, 4095])),
                          p.reshape(-1)[[5, 77, 4095]])
    assert np.array_equal(ds.noise_plane_t(small, 3).numpy(), p)
    v = ds.variance_scalars(cfg)
    assert 0.8 <= v.min() and v.max() <= 1.2 and abs(p.var() - v[3]) < 0.1


def test_tiny_scene_structure():
    cfg = ds.CONFIGS["tiny"]
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    assert sc.t.shape == (64,) and np.all(np.diff(sc.t) >= 0) and sc.t.max() <= 30.0
    assert np.allclose(np.linalg.norm(sc.obs_ecl, axis=1), 1.0) and np.all(sc.obs_ecl[:, 2] == 0)
    el = sc.elements()
    assert el.shape == (10000, 6) and list(sc.inj_index) == [5105]
    assert np.allclose(el[5105, :3], [2.7, 0.1, math.radians(5.0)], atol=1e-15)
    assert (sc.inj_pix[0, :, 0] >= 64).all() and (sc.inj_pix[0, :, 0] < 192).all()  # dither +-W/4
    f = sc.flux_plane_np(0)
    n = ds.noise_plane_np(cfg, 0)
    d = np.flatnonzero((f != n).reshape(-1))
    assert d.size == 1 and d[0] == sc.inj_pix[0, 0, 1] * 256 + sc.inj_pix[0, 0, 0]
    assert abs(float(f.reshape(-1)[d[0]] - n.reshape(-1)[d[0]]) - 0.5) < 1e-6
    assert np.array_equal(sc.flux_plane_t(0).numpy(), f)


def test_focused_variant_hits():
    cfg = ds.focused(ds.scaled(ds.CONFIGS["small_mba"], n_orbits=4000, n_exp=64, width=512,
                               height=512))
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    el = sc.elements()
    fam = ds.focus_mask(cfg, np.arange(4000))
    assert 0.4 < fam.mean() < 0.6
    pix = oracle.project(oracle.Survey.from_scene(sc), el, 0.0)["pix"]
    hits = (pix[..., 0] >= 0).sum(1)
    assert hits[fam].mean() > 2.0 and hits[~fam].sum() <= 2
    assert fam[sc.inj_index].all() and sc.inj_index.size == 100


def test_generators_hold_no_method_calls():
    """dtsynth must not import the oracle or the CUDA package (shared inputs only)."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for fn in ("rng.py", "workloads.py", "__init__.py"):
        tree = ast.parse(open(os.path.join(root, "dtsynth", fn)).read())
        for node in ast.walk(tree):
            names = []
            if isinstance(node, ast.Import):
                names = [a.name for a in node.names]
            elif isinstance(node, ast.ImportFrom):
                names = [node.module or ""]
            for nm in names:
                assert not nm.startswith("oracle") and "paper_2503_08854_b200" not in nm
