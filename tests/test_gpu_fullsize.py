"""GPU parity at BASELINE.json's FULL sizes (configs[1..4]) in the launch configuration bench.py times:
dt_stack over all candidate orbits against all exposures, then the oracle on SAMPLED outputs.

How a sample is checked without 134 GB of planes on the host: for the sampled orbits the oracle's own
projection gives the set H of exposures any of them hits; an orbit's sums only contain its hit
exposures, in ascending order, so the oracle evaluated on the sub-survey H (metadata and planes of
exactly those exposures, ascending) returns the same S, Wt, hits, SNR as on the full survey.  The
sample is the injected orbits, orbits the GPU reports hits for, and random candidates (mostly zero
hits: SNR = 0, hits = 0 must hold exactly).  Properties that hold at any size are checked on the whole
output: hit counts in [0, N], SNR finite, SNR = 0 where hits = 0, top-k equal to the oracle's top-k
of the same arrays.  Bars as in test_gpu_parity.py (hits exact, SNR within 1e-9 max(|SNR|, 1e-3) off
the 1e-6 px guard band).
"""
import numpy as np
import pytest

import dtsynth as ds
import oracle
from conftest import parity_record

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

HOST_PLANE_BYTES = 40 << 30    # planes of the oracle's sub-survey held on the host
N_RANDOM = 2000
N_HITTERS = 400
CHUNK = 5_000_000     # orbits generated per numpy call


def _dt():
    import paper_2503_08854_b200 as dt
    return dt


def _elements_device(cfg, dev):
    out = torch.empty((cfg.n_orbits, 6), dtype=torch.float64, device=dev)
    for lo in range(0, cfg.n_orbits, CHUNK):
        hi = min(cfg.n_orbits, lo + CHUNK)
        out[lo:hi] = torch.from_numpy(ds.elements(cfg, lo, hi)).to(dev)
    return out


def _var_plane_t(cfg, scene, j, dev):
    return torch.full((1, cfg.height, cfg.width), float(scene.var_scalar[j]), dtype=torch.float32, device=dev)


def _check_sample(cfg, scene, plane_of, snr, hits, sample, label):
    """Oracle on the sub-survey of the exposures the sampled orbits hit; plane_of(j) -> (flux, var) numpy."""
    el = np.concatenate([ds.elements(cfg, int(k), int(k) + 1) for k in sample])
    sv = oracle.Survey.from_scene(scene)
    pix = oracle.project(sv, el, scene.t0)["pix"]                  # [n, N, 2], (-1, -1) when culled
    hit = pix[..., 0] >= 0
    H_MAX = max(8, int(HOST_PLANE_BYTES // (cfg.plane_pixels * 4 * (2 if cfg.variance_mode == 1 else 1))))
    keep, H = [], set()
    for r in range(len(sample)):
        need = set(np.flatnonzero(hit[r]).tolist())
        if len(H | need) <= H_MAX:
            H |= need
            keep.append(r)
    keep = np.array(keep)
    Hs = np.array(sorted(H), dtype=np.int64)
    assert keep.size >= min(len(sample), N_RANDOM // 2), "sample collapsed"
    if Hs.size == 0:                                               # nobody hits anything
        Hs = np.array([0], dtype=np.int64)
    sub = oracle.Survey(scene.t[Hs], scene.obs_ecl[Hs], scene.ra0[Hs], scene.dec0[Hs], cfg.width, cfg.height,
                        scene.pixel_scale, scene.gm, scene.c, scene.obliquity, cfg.variance_mode,
                        scene.var_scalar[Hs])
    planes = [plane_of(int(j)) for j in Hs]
    ref = oracle.stack(sub, [p[0] for p in planes], [p[1] for p in planes] if cfg.variance_mode == 1 else None,
                       el[keep], scene.t0)
    idx = np.asarray(sample)[keep]
    g_snr, g_hits = snr[idx], hits[idx]
    clean = ref["nflag"] == 0
    assert np.array_equal(g_hits[clean], ref["hits"][clean]), label
    tol = 1e-9 * np.maximum(np.abs(ref["snr"]), 1e-3)
    ok = np.abs(g_snr - ref["snr"]) <= tol
    assert ok[clean].all(), (label, idx[~ok & clean][:10])
    flagged = np.flatnonzero(~clean)
    same = flagged[g_hits[flagged] == ref["hits"][flagged]]
    assert ok[same].all(), label
    assert (np.abs(g_hits - ref["hits"]) <= ref["nflag"]).all(), label   # at most one hit per flagged pair
    rep = dict(checked=int(keep.size), with_hits=int((ref["hits"] > 0).sum()), exposures=int(Hs.size),
                max_hits=int(ref["hits"].max()), flagged=int(flagged.size),
                flagged_hit_mismatch=int(flagged.size - same.size))
    parity_record("fullsize[%s]" % label, **rep)
    return rep


def _check_block_hit_counts(cfg, scene, hits, label, n_block=20000, lo=None):
    """A contiguous block of orbits, not chosen by the GPU's result: the oracle's projection gives every orbit's
    footprint hits over ALL exposures (the synthetic images carry no masked pixel, so that is the hit count); the
    GPU's counts must equal them exactly off the guard band and differ by at most the flagged pairs on it.  An orbit
    the GPU wrongly reports with zero (or too many) hits cannot hide behind the random sample."""
    lo = (cfg.n_orbits // 3) if lo is None else lo
    hi = min(cfg.n_orbits, lo + n_block)
    el = ds.elements(cfg, lo, hi)
    pr = oracle.project(oracle.Survey.from_scene(scene), el, scene.t0)
    want = (pr["pix"][..., 0] >= 0).sum(1)
    nflag = pr["flag"].astype(np.int64).sum(1)
    got = hits[lo:hi]
    clean = nflag == 0
    assert np.array_equal(got[clean], want[clean]), (label, np.flatnonzero(got[clean] != want[clean])[:10] + lo)
    assert (np.abs(got - want) <= nflag).all(), label
    rep = dict(block=[int(lo), int(hi)], pairs=int((hi - lo) * cfg.n_exp), oracle_hits=int(want.sum()),
               flagged_pairs=int(nflag.sum()), hit_count_mismatch_on_flagged=int((got != want).sum()))
    parity_record("fullsize_block[%s]" % label, **rep)
    return rep


def _pick_sample(scene, hits_dev, n):
    rng = np.random.default_rng(12345)
    rand = rng.integers(0, n, N_RANDOM)
    order = torch.nonzero(hits_dev > 0).flatten()
    if order.numel() > N_HITTERS:
        sel = torch.from_numpy(rng.choice(order.numel(), N_HITTERS, replace=False)).to(order.device)
        order = order[sel]
    hitters = order.cpu().numpy()
    inj = scene.inj_index[:200] if scene.inj_pix is not None else np.zeros(0, np.int64)
    allk = np.concatenate([inj.astype(np.int64), hitters.astype(np.int64), rand])   # hitters first
    _, first = np.unique(allk, return_index=True)
    return allk[np.sort(first)]


def _whole_output_properties(dt, trk, snr_dev, hits_dev, N):
    assert int(hits_dev.min()) >= 0 and int(hits_dev.max()) <= N
    assert bool(torch.isfinite(snr_dev).all())
    assert bool((snr_dev[hits_dev == 0] == 0).all())
    k = 64
    idx, val = trk.topk(k, min_hits=1)
    # the oracle's top-k over the same arrays (candidates: everything >= the k-th value keeps it cheap)
    cand = torch.nonzero((hits_dev >= 1) & (snr_dev >= float(val[-1]) if len(val) else hits_dev >= 1)).flatten()
    cs, ch = snr_dev[cand].cpu().numpy(), hits_dev[cand].cpu().numpy()
    widx, wval = oracle.topk(cs, ch, k, 1)
    assert np.array_equal(cand.cpu().numpy()[widx], idx) and np.array_equal(wval, val)


RESIDENT = ["small_mba", "small_mba+focused", "neo", "neo+focused", "tno", "tno+focused"]


@pytest.mark.parametrize("name", RESIDENT)
def test_full_size_resident(name):
    """configs[1], [3], [4]: images resident in HBM, all candidate orbits in one dt_stack call."""
    dt = _dt()
    dev = torch.device("cuda", 0)
    cfg = ds.CONFIGS[name.split("+")[0]]
    if name.endswith("+focused"):
        cfg = ds.focused(cfg)
    need = cfg.image_bytes() + cfg.n_orbits * (48 + 36 + 12) + (6 << 30)
    free, _total = torch.cuda.mem_get_info()
    if free < need:
        pytest.skip("needs %.0f GB of free HBM" % (need / 1e9))
    scene = ds.build_scene(cfg, oracle.scene_project_fn)
    with dt.Tracker.from_scene(scene, hbm_budget_bytes=cfg.image_bytes() + (1 << 30)) as trk:
        for j in range(cfg.n_exp):
            f = scene.flux_plane_t(j, dev).unsqueeze(0).contiguous()
            v = _var_plane_t(cfg, scene, j, dev) if cfg.variance_mode == 1 else None
            trk.load_image_batch(j, f, v)
        del f, v
        el = _elements_device(cfg, dev)
        snr, hits = trk.stack(el, scene.t0)
        st = trk.stats()
        assert st["streamed"] == 0 and st["pairs"] == cfg.pairs and st["invalid_orbits"] == 0
        assert int(hits.sum(dtype=torch.int64)) == st["hits"]
        _whole_output_properties(dt, trk, snr, hits, cfg.n_exp)
        sample = _pick_sample(scene, hits, cfg.n_orbits)
        snr_h, hits_h = snr.cpu().numpy(), hits.cpu().numpy()

        def plane_of(j):
            fl = scene.flux_plane_t(j, dev).cpu().numpy()
            return fl, (np.full_like(fl, np.float32(scene.var_scalar[j])) if cfg.variance_mode == 1 else None)

        rep = _check_sample(cfg, scene, plane_of, snr_h, hits_h, sample, name)
        blk = _check_block_hit_counts(cfg, scene, hits_h, name)
        if name.endswith("+focused"):
            assert blk["oracle_hits"] > 1000, "vacuous block"
        print(name, blk)
        print(name, "pairs %.3g hits %d ms %.1f" % (cfg.pairs, st["hits"], st["ms_total"]), rep)
        if name.endswith("+focused"):
            assert rep["with_hits"] > 0
            # injected-source recovery in aggregate: z = SNR - A sum(1/sigma)/sqrt(sum 1/sigma^2)
            if scene.inj_pix is not None:
                hitmask = scene.inj_pix[..., 0] >= 0
                w = 1.0 / np.sqrt(scene.var_scalar)
                expect = scene.inj_amp * (hitmask * w * np.sqrt(scene.var_scalar) * w).sum(1) / \
                    np.sqrt(np.maximum((hitmask * w * w).sum(1), 1e-300))
                sel = hitmask.sum(1) >= 8
                z = snr_h[scene.inj_index[sel]] - expect[sel]
                if sel.sum() >= 30:
                    print("  injected sources with >= 8 hits: %d, z mean %.3f sd %.3f" % (sel.sum(), z.mean(), z.std()))
                    assert abs(z.mean()) < 6.0 / np.sqrt(sel.sum()) + 0.1, z.mean()
                    assert 0.6 < z.std() < 1.4, z.std()


def test_full_size_lsst_streamed():
    """configs[2]: 2000 exposures of 4096x4096 flux + variance = 268 GB > HBM, streamed in double-buffered
    batches from pinned host memory.  The host holds a pool of POOL distinct seeded exposures and exposure
    j streams pool[j mod POOL] (SURVEY.md 8(d) "Host memory"): the bytes moved are the full 268 GB."""
    dt = _dt()
    dev = torch.device("cuda", 0)
    cfg = ds.CONFIGS["lsst"]
    POOL = 64
    plane_b = cfg.plane_pixels * 4
    import psutil
    if psutil.virtual_memory().available < 2 * POOL * plane_b + (16 << 30):
        pytest.skip("needs %.0f GB of host memory for the pinned pool" % (2 * POOL * plane_b / 1e9))
    scene = ds.build_scene(cfg, None, inject=False)        # pooled planes cannot carry per-exposure sources
    # exposure j carries pool[j % POOL]: variance must follow the plane
    scene.var_scalar = scene.var_scalar[np.arange(cfg.n_exp) % POOL].copy()
    flux_pool = torch.empty((POOL, cfg.height, cfg.width), dtype=torch.float32).pin_memory()
    var_pool = torch.empty((POOL, cfg.height, cfg.width), dtype=torch.float32).pin_memory()
    for q in range(POOL):
        flux_pool[q].copy_(ds.noise_plane_t(cfg, q, dev))
        var_pool[q].fill_(float(scene.var_scalar[q]))
    el = _elements_device(cfg, dev)
    results = {}
    for mode in ("0", "-1"):      # streamed batch by batch, then the library's own choice (zero-copy gather)
        if True:
            with dt.Tracker.from_scene(scene) as trk:
                trk.set_option("stream_zero_copy", int(mode))
                trk.set_option("stream_tiles", 0)       # mode 0: whole planes in double-buffered batches
                for j in range(cfg.n_exp):
                    trk.load_image_batch(j, flux_pool[j % POOL:j % POOL + 1], var_pool[j % POOL:j % POOL + 1])
                snr, hits = trk.stack(el, scene.t0)
                st = trk.stats()
                assert st["streamed"] == 1 and st["n_image_batches"] >= 2
                if mode == "0":
                    assert st["image_zero_copy"] == 0 and st["h2d_image_bytes"] == cfg.image_bytes()
                else:
                    assert st["image_zero_copy"] == 1 and st["h2d_image_bytes"] == 0   # 6.8e4 hits: no image is copied
                _whole_output_properties(dt, trk, snr, hits, cfg.n_exp)
                results[mode] = (snr.cpu().numpy(), hits.cpu().numpy(), st)
                if mode == "0":
                    sample = _pick_sample(scene, hits, cfg.n_orbits)
    assert np.array_equal(results["0"][0], results["-1"][0]) and np.array_equal(results["0"][1], results["-1"][1])
    snr_h, hits_h, st = results["0"]

    def plane_of(j):
        return flux_pool[j % POOL].numpy(), var_pool[j % POOL].numpy()

    rep = _check_sample(cfg, scene, plane_of, snr_h, hits_h, sample, "lsst streamed")
    _check_block_hit_counts(cfg, scene, hits_h, "lsst streamed", n_block=10000)
    gbs = st["h2d_image_bytes"] / (st["ms_total"] * 1e-3) * 1e-9
    print("lsst streamed: pairs %.3g hits %d ms %.0f (%.1f GB/s host->device); zero-copy gather: ms %.0f (%.3g pairs/s)" %
          (cfg.pairs, st["hits"], st["ms_total"], gbs, results["-1"][2]["ms_total"],
           cfg.pairs / (results["-1"][2]["ms_total"] * 1e-3)), rep)
