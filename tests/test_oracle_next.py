"""Pins (P11) of the oracle's SURVEY.md 8(f) NEXT rows: dto_stack_ex (patch gather with PSF weights, PAPER.md:143;
per-intersection outlier rejection; per-orbit epochs) and dto_threshold (Alg. 1
`FindSignificantResults`).  The paper gives prose only (readings A21-A24 in DESIGN.md), so
the pins are: reduction to the already pinned dto_stack, closed forms on flat images, an independent numpy
brute force (including patches cut by the footprint edge and masked pixels), the two-body identity
M0(t0 + D) = M0(t0) + n D for the epochs, and numpy for the threshold.  All CPU.
"""
import math

import numpy as np

import dtsynth as ds
import oracle

GM = ds.GM_SUN


def _scene(n_orb=300, n_exp=20, W=64, H=48, mode=1):
    cfg = ds.focused(ds.scaled(ds.CONFIGS["tiny"], n_orbits=n_orb, n_exp=n_exp, width=W, height=H,
                               variance_mode=mode, var_range=(0.8, 1.2)))
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    flux = [sc.flux_plane_np(j) for j in range(n_exp)]
    var = [sc.var_plane_np(j) for j in range(n_exp)] if mode == 1 else None
    return sc, oracle.Survey.from_scene(sc), flux, var


def test_p11_patch1_unit_weight_is_the_plain_stack_bit_for_bit():
    for mode in (0, 1):
        sc, sv, flux, var = _scene(mode=mode)
        el = sc.elements()
        a = oracle.stack(sv, flux, var, el, sc.t0)
        b = oracle.stack_ex(sv, flux, var, el, sc.t0, patch=1, weights=[1.0])
        c = oracle.stack_ex(sv, flux, var, el, sc.t0, patch=1, t0_per_orbit=np.full(el.shape[0], sc.t0))
        assert a["hits"].sum() > 100
        for key in ("snr", "hits", "S", "Wt", "nflag"):
            assert np.array_equal(a[key], b[key]), key
            assert np.array_equal(a[key], c[key]), key


def _brute(sc, sv, flux, var, el, k, w, clip):
    """Independent evaluation of the definition from the oracle's PIXEL INDICES only (numpy, own loops)."""
    pix = oracle.project(sv, el, sc.t0)["pix"]
    H, W = flux[0].shape
    h = k // 2
    w = np.asarray(w, float).reshape(k, k)
    S, Wt, hits = np.zeros(len(el)), np.zeros(len(el)), np.zeros(len(el), np.int32)
    for o in range(len(el)):
        for j in range(len(flux)):
            ix, iy = pix[o, j]
            if ix < 0:
                continue
            si = wti = 0.0
            used = 0
            for dy in range(-h, h + 1):
                for dx in range(-h, h + 1):
                    y, x = iy + dy, ix + dx
                    if not (0 <= y < H and 0 <= x < W):
                        continue
                    f = np.float64(flux[j][y, x])
                    v = np.float64(var[j][y, x]) if var is not None else sv.var_scalar[j]
                    if not (np.isfinite(f) and np.isfinite(v) and v > 0):
                        continue
                    si += (w[dy + h, dx + h] * f) / v
                    wti += (w[dy + h, dx + h] ** 2) / v
                    used += 1
            if used == 0 or si > clip * math.sqrt(wti):
                continue
            S[o] += si
            Wt[o] += wti
            hits[o] += 1
    snr = np.where(hits > 0, S / np.sqrt(np.where(Wt > 0, Wt, 1.0)), 0.0)
    return snr, hits, S, Wt


def test_p11_patch_brute_force_with_edges_masks_and_clip():
    rng = np.random.default_rng(3)
    for mode, k, clip in [(1, 3, math.inf), (0, 5, math.inf), (1, 3, 1.5), (0, 1, 0.7)]:
        sc, sv, flux, var = _scene(n_orb=200, n_exp=16, W=40, H=32, mode=mode)
        flux = [f.copy() for f in flux]
        for f in flux:                                     # masked pixels, and a bright outlier or two
            f.reshape(-1)[rng.integers(0, f.size, 40)] = np.nan
            f.reshape(-1)[rng.integers(0, f.size, 10)] = 50.0
        if var is not None:
            var = [v.copy() for v in var]
            var[3].reshape(-1)[rng.integers(0, var[3].size, 30)] = 0.0
        w = rng.uniform(0.1, 1.0, (k, k))
        el = sc.elements()
        ref = oracle.stack_ex(sv, flux, var, el, sc.t0, patch=k, weights=w, clip=clip)
        snr, hits, S, Wt = _brute(sc, sv, flux, var, el, k, w, clip)
        assert hits.sum() > 50
        assert np.array_equal(ref["hits"], hits)
        assert np.array_equal(ref["S"], S) and np.array_equal(ref["Wt"], Wt)      # same operations, same order
        assert np.allclose(ref["snr"], snr, rtol=0, atol=1e-15)
        # hits on the footprint edge exist in this scene (patches cut by the edge are exercised)
        pix = oracle.project(sv, el, sc.t0)["pix"]
        edge = (pix[..., 0] == 0) | (pix[..., 1] == 0) | (pix[..., 0] == 39) | (pix[..., 1] == 31)
        assert edge.any()
        if math.isfinite(clip):
            plain = oracle.stack_ex(sv, flux, var, el, sc.t0, patch=k, weights=w)
            assert (plain["hits"] >= ref["hits"]).all() and (plain["hits"] > ref["hits"]).any()


def test_p11_flat_image_closed_form():
    """f = c, v = s2 everywhere, every patch inside the image: s_i = c sum(w) / s2, wt_i = sum(w^2) / s2, so
    SNR = c sum(w) sqrt(hits) / sqrt(s2 sum(w^2)); equal weights recover c k sqrt(hits / s2)."""
    sc, sv, _, _ = _scene(n_orb=200, n_exp=12, W=64, H=64, mode=1)
    c, s2, k = 0.75, 2.0, 3
    flux = [np.full((64, 64), c, np.float32)] * 12
    var = [np.full((64, 64), s2, np.float32)] * 12
    w = np.array([[0.05, 0.1, 0.05], [0.1, 0.4, 0.1], [0.05, 0.1, 0.05]])
    el = sc.elements()
    pix = oracle.project(sv, el, sc.t0)["pix"]
    hit = pix[..., 0] >= 0
    interior = (~hit | ((pix[..., 0] >= 1) & (pix[..., 0] <= 62) & (pix[..., 1] >= 1) & (pix[..., 1] <= 62))).all(1)
    ref = oracle.stack_ex(sv, flux, var, el, sc.t0, patch=k, weights=w)
    n = hit.sum(1)
    want = c * w.sum() * np.sqrt(n) / math.sqrt(s2 * (w ** 2).sum())
    sel = interior & (n > 0)
    assert sel.sum() > 20
    assert np.array_equal(ref["hits"][sel], n[sel])
    assert np.allclose(ref["snr"][sel], want[sel], rtol=1e-13)
    eq = oracle.stack_ex(sv, flux, var, el, sc.t0, patch=k)              # weights NULL = all 1
    assert np.allclose(eq["snr"][sel], c * k * np.sqrt(n[sel] / s2), rtol=1e-13)


def test_p11_clip_is_one_sided_and_strict():
    """Unit images: every intersection has s_i = 1, wt_i = 1 (per-intersection SNR exactly 1)."""
    sc, sv, _, _ = _scene(n_orb=100, n_exp=10, mode=1)
    one = [np.ones((48, 64), np.float32)] * 10
    el = sc.elements()
    base = oracle.stack_ex(sv, one, one, el, sc.t0)
    assert base["hits"].max() > 0
    assert np.array_equal(oracle.stack_ex(sv, one, one, el, sc.t0, clip=1.0)["hits"], base["hits"])   # 1 > 1 is false
    none = oracle.stack_ex(sv, one, one, el, sc.t0, clip=0.999)
    assert (none["hits"] == 0).all() and (none["snr"] == 0).all()
    neg = [-p for p in one]                                                # anomalously LOW is kept (one-sided)
    assert np.array_equal(oracle.stack_ex(sv, neg, one, el, sc.t0, clip=0.5)["hits"], base["hits"])
    # one bright pixel on the path of one orbit: exactly that intersection goes
    pix = oracle.project(sv, el, sc.t0)["pix"]
    o = int(np.argmax(base["hits"]))
    j = int(np.flatnonzero(pix[o, :, 0] >= 0)[0])
    planes = [p.copy() for p in one]
    planes[j][pix[o, j, 1], pix[o, j, 0]] = 30.0
    cl = oracle.stack_ex(sv, planes, one, el, sc.t0, clip=5.0)
    assert cl["hits"][o] == base["hits"][o] - 1
    assert cl["snr"][o] == math.sqrt(base["hits"][o] - 1) or abs(cl["snr"][o] - math.sqrt(base["hits"][o] - 1)) < 1e-15


def test_p11_epoch_shift_identity():
    """Two-body motion: elements (.., M0) at epoch t0 and (.., M0 + n D) at epoch t0 + D are the same orbit
    (n = sqrt(GM / a^3)), so per-orbit epochs D_o with shifted M0 must reproduce the scalar-epoch result
    (up to the rounding of M: hit sets equal off the guard band, SNR to 1e-9)."""
    sc, sv, flux, var = _scene(n_orb=300, n_exp=20, mode=1)
    el = sc.elements()
    rng = np.random.default_rng(11)
    D = rng.uniform(-400.0, 400.0, el.shape[0])
    el2 = el.copy()
    el2[:, 5] = el[:, 5] + np.sqrt(GM / el[:, 0] ** 3) * D
    a = oracle.stack_ex(sv, flux, var, el, sc.t0)
    b = oracle.stack_ex(sv, flux, var, el2, 123.0, t0_per_orbit=sc.t0 + D)       # the scalar is ignored
    clean = (a["nflag"] == 0) & (b["nflag"] == 0)
    assert clean.sum() > 250 and a["hits"][clean].sum() > 100
    assert np.array_equal(a["hits"][clean], b["hits"][clean])
    assert np.allclose(a["snr"][clean], b["snr"][clean], rtol=0, atol=1e-9)
    # a wrong epoch is a different orbit: shifting the epoch WITHOUT shifting M0 loses the hits
    c = oracle.stack_ex(sv, flux, var, el, sc.t0, t0_per_orbit=sc.t0 + 30.0 + 0 * D)
    assert c["hits"].sum() < 0.2 * a["hits"].sum()
    # invalid epoch -> invalid orbit
    bad = np.full(el.shape[0], sc.t0)
    bad[7] = np.nan
    d = oracle.stack_ex(sv, flux, var, el, sc.t0, t0_per_orbit=bad)
    assert d["hits"][7] == -1 and np.isnan(d["snr"][7]) and np.array_equal(d["hits"][8:], a["hits"][8:])


def test_p11_threshold_equals_numpy():
    rng = np.random.default_rng(5)
    snr = rng.normal(0, 3, 5000)
    snr[rng.integers(0, 5000, 50)] = np.nan
    snr[17] = 5.0
    hits = rng.integers(-1, 6, 5000).astype(np.int32)
    for snr_min, min_hits in [(5.0, 0), (5.0, 3), (-1.0, 1), (100.0, 0)]:
        want = np.flatnonzero(np.isfinite(snr) & (snr >= snr_min) & (hits >= min_hits))
        idx, val, nf = oracle.threshold(snr, hits, snr_min, min_hits)
        assert nf == want.size and np.array_equal(idx, want) and np.array_equal(val, snr[want])
        idx2, _, nf2 = oracle.threshold(snr, hits, snr_min, min_hits, max_out=3)       # truncated output, full count
        assert nf2 == want.size and np.array_equal(idx2, want[:3])
    assert 17 in oracle.threshold(snr, hits, 5.0, -1)[0]                               # >= is inclusive
