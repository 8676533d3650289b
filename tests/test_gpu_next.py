"""GPU parity of the SURVEY.md 8(f) NEXT rows against the oracle's dto_stack_ex / dto_threshold, through the C ABI:
NEXT-1 patch gather (dt_set_patch), NEXT-3 per-intersection outlier rejection
(dt_set_outlier_clip), per-orbit epochs (dt_stack_epochs) and threshold mode
(dt_threshold).  Bars as everywhere: hit counts exact off the 1e-6 px guard band, SNR within
1e-9 max(|SNR|, 1e-3); the sums use the definition's operations in the definition's order, so on orbits whose hit
sets agree SNR is expected to be bit-identical (counted and recorded)."""
import math

import numpy as np
import pytest

import dtsynth as ds
import oracle
from conftest import parity_record

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _dt():
    import paper_2503_08854_b200 as dt
    return dt


def _scene(base, focused=True, **kw):
    cfg = ds.scaled(ds.CONFIGS[base], **kw)
    if focused:
        cfg = ds.focused(cfg)
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    N = cfg.n_exp
    flux = np.stack([sc.flux_plane_np(j) for j in range(N)])
    var = np.stack([sc.var_plane_np(j) for j in range(N)]) if cfg.variance_mode == 1 else None
    return sc, flux, var


def _compare(snr, hits, ref, what):
    snr, hits = np.asarray(snr), np.asarray(hits)
    clean = ref["nflag"] == 0
    assert np.array_equal(hits[clean], ref["hits"][clean]), what
    tol = 1e-9 * np.maximum(np.abs(ref["snr"]), 1e-3)
    ok = (np.isnan(snr) & np.isnan(ref["snr"])) | (np.abs(snr - ref["snr"]) <= tol)
    assert ok[clean].all(), (what, np.flatnonzero(~ok & clean)[:10])
    valid = ref["hits"] >= 0
    assert (np.abs(hits - ref["hits"])[valid] <= ref["nflag"][valid]).all(), what
    same = clean & (hits == ref["hits"])
    parity_record("next[%s]" % what, orbits=int(hits.size), flagged_orbits=int((~clean).sum()),
                  hits=int(ref["hits"][valid].sum()), snr_bit_identical=int((snr[same] == ref["snr"][same]).sum()),
                  compared=int(same.sum()))
    assert ref["hits"][valid].sum() > 100, "vacuous"


CASES = {
    "mba_scalar_var": ("small_mba", dict(n_orbits=5003, n_exp=70, width=256, height=192)),
    "tno_plane_var": ("tno", dict(n_orbits=4000, n_exp=90, width=320, height=256)),
    "tiny_edges": ("tiny", dict(n_orbits=3000, n_exp=40, width=48, height=40)),     # patches cut by the footprint edge
}


@pytest.mark.parametrize("k", [1, 3, 5])
@pytest.mark.parametrize("case", list(CASES))
def test_patch_gather_parity(case, k):
    dt = _dt()
    base, kw = CASES[case]
    sc, flux, var = _scene(base, **kw)
    rng = np.random.default_rng(17 + k)
    flux = flux.copy()
    flux.reshape(-1)[rng.integers(0, flux.size, flux.size // 500)] = np.nan          # masked pixels
    if var is not None:
        var = var.copy()
        var.reshape(-1)[rng.integers(0, var.size, var.size // 1000)] = 0.0
    # a PSF-like kernel: Gaussian, sigma 0.8 px, normalised (any weights would do)
    ax = np.arange(k) - k // 2
    w = np.exp(-0.5 * (ax[:, None] ** 2 + ax[None, :] ** 2) / 0.8 ** 2)
    w /= w.sum()
    el = sc.elements()
    sv = oracle.Survey.from_scene(sc)
    ref = oracle.stack_ex(sv, list(flux), list(var) if var is not None else None, el, sc.t0, patch=k, weights=w)
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux, var)
        trk.set_patch(k, w)
        snr, hits = trk.stack(el, sc.t0)
        _compare(snr, hits, ref, "patch k=%d %s" % (k, case))
        if k == 1:
            # k = 1 with unit weight IS the single-pixel stack: same bits as the plain path of the library
            trk.set_patch(1, None)
            snr1, hits1 = trk.stack(el, sc.t0)
            w1 = float(w[0, 0])
            assert w1 == 1.0 and np.array_equal(hits1, hits) and np.array_equal(snr1, snr, equal_nan=True)
        # equal weights through the NULL pointer
        trk.set_patch(k, None)
        snr_e, hits_e = trk.stack(el, sc.t0)
        ref_e = oracle.stack_ex(sv, list(flux), list(var) if var is not None else None, el, sc.t0, patch=k)
        _compare(snr_e, hits_e, ref_e, "patch k=%d equal weights %s" % (k, case))
    if case == "tiny_edges":
        pix = oracle.project(sv, el, sc.t0)["pix"]
        assert ((pix[..., 0] == 0) | (pix[..., 1] == 0) | (pix[..., 0] == 47) | (pix[..., 1] == 39)).any()


@pytest.mark.parametrize("case,k,clip", [("mba_scalar_var", 1, 1.5), ("tno_plane_var", 1, 2.0), ("tno_plane_var", 3, 1.0),
                                         ("mba_scalar_var", 3, 0.0)])
def test_outlier_clip_parity(case, k, clip):
    dt = _dt()
    base, kw = CASES[case]
    sc, flux, var = _scene(base, **kw)
    el = sc.elements()
    sv = oracle.Survey.from_scene(sc)
    args = (sv, list(flux), list(var) if var is not None else None, el, sc.t0)
    ref = oracle.stack_ex(*args, patch=k, clip=clip)
    plain = oracle.stack_ex(*args, patch=k)
    assert plain["hits"].sum() > ref["hits"].sum() > 0, "the clip must reject some intersections and keep some"
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux, var)
        trk.set_patch(k, None)
        trk.set_outlier_clip(clip)
        snr, hits = trk.stack(el, sc.t0)
        _compare(snr, hits, ref, "clip %.1f k=%d %s" % (clip, k, case))
        trk.set_outlier_clip(math.inf)
        snr, hits = trk.stack(el, sc.t0)
        _compare(snr, hits, plain, "clip off k=%d %s" % (k, case))
        with pytest.raises(dt.DtError):
            trk.set_outlier_clip(math.nan)


def test_per_orbit_epochs_parity():
    dt = _dt()
    base, kw = CASES["mba_scalar_var"]
    sc, flux, var = _scene(base, **kw)
    el = sc.elements().copy()
    n = el.shape[0]
    rng = np.random.default_rng(23)
    D = rng.uniform(-300.0, 300.0, n)
    el[:, 5] += np.sqrt(ds.GM_SUN / el[:, 0] ** 3) * D          # same orbits, expressed at other epochs
    t0 = sc.t0 + D
    t0[5] = np.nan                                              # invalid epoch -> invalid orbit
    sv = oracle.Survey.from_scene(sc)
    ref = oracle.stack_ex(sv, list(flux), None, el, 0.0, t0_per_orbit=t0)
    assert ref["hits"][5] == -1
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux, var)
        snr, hits = trk.stack(el, t0)                           # numpy epochs -> dt_stack_epochs
        _compare(snr, hits, ref, "epochs host")
        assert hits[5] == -1 and np.isnan(snr[5]) and trk.stats()["invalid_orbits"] == 1
        snr_d, hits_d = trk.stack(torch.from_numpy(el).cuda(), torch.from_numpy(t0).cuda())
        assert np.array_equal(hits_d.cpu().numpy(), hits) and np.array_equal(snr_d.cpu().numpy(), snr, equal_nan=True)
        # the same orbits at the scalar epoch: same hit sets off the guard band
        plain = oracle.stack(sv, list(flux), None, sc.elements(), sc.t0)
        clean = (plain["nflag"] == 0) & (ref["nflag"] == 0)
        clean[5] = False
        assert np.array_equal(plain["hits"][clean], hits[clean])


def test_threshold_mode():
    dt = _dt()
    base, kw = CASES["tno_plane_var"]
    sc, flux, var = _scene(base, **kw)
    el = sc.elements()
    with dt.Tracker.from_scene(sc) as trk:
        with pytest.raises(dt.DtError):
            trk.threshold(5.0)                                  # no result yet
        trk.load_image_batch(0, flux, var)
        snr, hits = trk.stack(el, sc.t0)
        for snr_min, min_hits, max_out in [(5.0, 0, 1 << 20), (1.0, 3, 1 << 20), (0.0, 0, 1 << 20), (-1e300, 1, 7),
                                           (1e300, 0, 10), (float(np.sort(snr)[-5]), 0, 100), (2.0, 0, 0)]:
            idx, val, nf = trk.threshold(snr_min, min_hits, max_out)
            widx, wval, wnf = oracle.threshold(snr, hits, snr_min, min_hits, max_out)
            assert nf == wnf and np.array_equal(idx, widx) and np.array_equal(val, wval), (snr_min, min_hits, max_out)
        assert trk.threshold(float(np.sort(snr)[-5]))[2] >= 5   # >= is inclusive
        with pytest.raises(dt.DtError):
            trk.threshold(math.nan)


def test_patch_through_the_zero_copy_gather():
    """Streaming mode, few hits: the extended stack reads the patch straight from the page-locked host planes."""
    dt = _dt()
    base, kw = CASES["tno_plane_var"]
    sc, flux, var = _scene(base, **kw)
    el = sc.elements()
    w = np.array([[0.0, 0.2, 0.0], [0.2, 1.0, 0.2], [0.0, 0.2, 0.0]])
    ref = oracle.stack_ex(oracle.Survey.from_scene(sc), list(flux), list(var), el, sc.t0, patch=3, weights=w, clip=3.0)
    pf, pv = torch.from_numpy(flux).pin_memory(), torch.from_numpy(var).pin_memory()
    for zero_copy in (0, 1):
        with dt.Tracker.from_scene(sc, hbm_budget_bytes=2 * 20 * flux[0].nbytes * 2) as trk:
            trk.set_option("stream_zero_copy", zero_copy)
            trk.load_image_batch(0, pf, pv)
            trk.set_patch(3, w)
            trk.set_outlier_clip(3.0)
            snr, hits = trk.stack(el, sc.t0)
            assert trk.stats()["image_zero_copy"] == zero_copy
            _compare(snr, hits, ref, "patch 3 clip 3 streamed zero_copy=%d" % zero_copy)


def test_exposure_sharded_partial_sums():
    """SURVEY 8(f) NEXT-4 on one GPU: two contexts on the two halves of the exposures stand for two ranks (no rank
    waits on another: the lists are handed over in-process; the all-gather itself is tested with gloo in
    tests/test_sharded_gloo.py).  Each compacts its sparse per-orbit sums on the device; adding the lists in rank order
    on either context gives, bit for bit, the oracle's sums of the two slices added in that order, the plain stack's
    hit counts, and its SNR to the rounding of a re-associated sum; top-k and threshold see the merged result."""
    dt = _dt()
    from paper_2503_08854_b200.sharded import exposure_slices
    base, kw = CASES["mba_scalar_var"]
    sc, flux, var = _scene(base, **kw)
    el = sc.elements().copy()
    el[3, 1] = 1.5                                               # one invalid orbit
    n, N = el.shape[0], sc.cfg.n_exp
    sv = oracle.Survey.from_scene(sc)
    full = oracle.stack(sv, list(flux), None, el, sc.t0)
    slices = exposure_slices(N, 2)
    ref_S, ref_W, ref_h = np.zeros(n), np.zeros(n), np.zeros(n, np.int64)
    for lo, hi in slices:                                        # the sharded definition, from the oracle
        sub = oracle.Survey(sc.t[lo:hi], sc.obs_ecl[lo:hi], sc.ra0[lo:hi], sc.dec0[lo:hi], sc.cfg.width, sc.cfg.height,
                            sc.pixel_scale, sc.gm, sc.c, sc.obliquity, 0, sc.var_scalar[lo:hi])
        r = oracle.stack(sub, list(flux[lo:hi]), None, el, sc.t0)
        ok = r["hits"] > 0
        ref_S[ok] += r["S"][ok]
        ref_W[ok] += r["Wt"][ok]
        ref_h[ok] += r["hits"][ok]
    el_dev = torch.from_numpy(el).cuda()
    trks, lists = [], []
    try:
        for (lo, hi) in slices:
            t = dt.Tracker(sc.t[lo:hi], sc.obs_ecl[lo:hi], sc.ra0[lo:hi], sc.dec0[lo:hi], sc.cfg.width, sc.cfg.height,
                           sc.pixel_scale, gm=sc.gm, c=sc.c, obliquity=sc.obliquity, variance_mode=0,
                           var_scalar=sc.var_scalar[lo:hi])
            t.load_image_batch(0, flux[lo:hi])
            t.stack(el_dev, sc.t0)
            trks.append(t)
            lists.append(dt.dt_partials_sparse(t.ctx, n, device=el_dev.device))
        assert all(0 < int(p[0].numel()) < n for p in lists), "sparse lists"
        assert all(bool((p[0][1:] > p[0][:-1]).all()) for p in lists), "index ascending"
        results = []
        for t in trks:                                           # every "rank" merges all lists in rank order
            dt.dt_partials_reset(t.ctx)
            for part in lists:
                dt.dt_partials_add(t.ctx, *part)
            snr, hits = dt.dt_partials_finalize(t.ctx, n, device=el_dev.device)
            results.append((snr.cpu().numpy(), hits.cpu().numpy()))
        assert np.array_equal(results[0][0], results[1][0], equal_nan=True) and np.array_equal(results[0][1], results[1][1])
        snr, hits = results[0]
        clean = full["nflag"] == 0
        assert hits[3] == -1 and np.isnan(snr[3])
        assert np.array_equal(hits[clean], full["hits"][clean])
        want = np.where(ref_h > 0, ref_S / np.sqrt(np.where(ref_W > 0, ref_W, 1.0)), 0.0)
        same = clean & (hits == ref_h) & (hits >= 0)
        assert same.sum() > n // 2 and np.array_equal(snr[same], want[same]), "the sharded definition, bit for bit"
        assert np.all(np.abs(snr - full["snr"])[clean & (hits >= 0)] <= 1e-9 * np.maximum(np.abs(full["snr"]), 1e-3)[clean & (hits >= 0)])
        idx, val = trks[0].topk(5, min_hits=1)
        widx, wval = oracle.topk(snr, hits, 5, 1)
        assert np.array_equal(idx, widx) and np.array_equal(val, wval)
        # host lists work too, and a bad index is refused
        dt.dt_partials_reset(trks[0].ctx)
        for part in lists:
            dt.dt_partials_add(trks[0].ctx, *[x.cpu().numpy() for x in part])
        snr_h, hits_h = dt.dt_partials_finalize(trks[0].ctx, n)
        assert np.array_equal(snr_h, snr, equal_nan=True) and np.array_equal(hits_h, hits)
        with pytest.raises(dt.DtError):
            dt.dt_partials_add(trks[0].ctx, np.array([n], np.int64), np.ones(1), np.ones(1), np.ones(1, np.int32))
        parity_record("next[sharded x2]", orbits=n, flagged_orbits=int((~clean).sum()), hits=int(ref_h.sum()),
                      snr_bit_identical=int(same.sum()), compared=int(same.sum()),
                      list_lengths=[int(p[0].numel()) for p in lists])
    finally:
        for t in trks:
            t.close()
