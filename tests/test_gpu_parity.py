"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle on the
same seeded inputs.  Bars (BASELINE.json north_star):
  * sky positions within 1e-10 rad;
  * pixel indices bit-exact except where the oracle flags the fractional coordinate within 1e-6 px
    of a rounding boundary (A11) -- such cases are counted and reported;
  * per-orbit hits exact and SNR within 1e-9 * max(|SNR|, 1e-3) (A14) on orbits without flagged hits.
Sizes: small enough for the oracle to finish in seconds, large enough to span several 256-orbit
tiles, several 32-exposure groups, ragged tails in both, and more than one work unit.
"""
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


def _planes(sc, mode):
    N = sc.cfg.n_exp
    flux = np.stack([sc.flux_plane_np(j) for j in range(N)])
    var = np.stack([sc.var_plane_np(j) for j in range(N)]) if mode == 1 else None
    return flux, var


def _compare_stack(snr, hits, ref, what=""):
    snr, hits = np.asarray(snr), np.asarray(hits)
    clean = ref["nflag"] == 0
    assert np.array_equal(hits[clean], ref["hits"][clean]), what
    tol = 1e-9 * np.maximum(np.abs(ref["snr"]), 1e-3)
    both_nan = np.isnan(snr) & np.isnan(ref["snr"])
    ok = both_nan | (np.abs(snr - ref["snr"]) <= tol)
    assert ok[clean].all(), (what, np.flatnonzero(~ok & clean)[:10])
    flagged = np.flatnonzero(~clean)
    same = flagged[hits[flagged] == ref["hits"][flagged]]
    assert ok[same].all(), what
    # an orbit with k flagged pairs may differ from the oracle by at most k hits (each flagged pair may
    # fall on either side of its rounding boundary or footprint edge), never by more
    valid = ref["hits"] >= 0
    assert (np.abs(hits - ref["hits"])[valid] <= ref["nflag"][valid]).all(), what
    rep = dict(orbits=int(hits.size), flagged_orbits=int(flagged.size), flagged_hit_mismatch=int(flagged.size - same.size),
               hits=int(ref["hits"][valid].sum()))
    if what:
        parity_record("stack[%s]" % what, **rep)
    return rep


def _compare_project(out, ref):
    """-> number of pixel mismatches inside the guard band (reported); asserts the rest."""
    valid = np.isfinite(ref["radec"][..., 0])
    dra = np.abs(out["radec"][..., 0] - ref["radec"][..., 0])
    dra = np.minimum(dra, 2 * math.pi - dra)
    cosd = np.cos(ref["radec"][..., 1])
    assert (dra[valid] * cosd[valid]).max() <= 1e-10          # great-circle east-west offset
    assert np.abs(out["radec"][..., 1] - ref["radec"][..., 1])[valid].max() <= 1e-10
    same = (out["pix"] == ref["pix"]).all(-1)
    bad = ~same
    assert not (bad & (ref["flag"] == 0)).any(), np.argwhere(bad & (ref["flag"] == 0))[:5]
    # continuous pixel coordinates, where the projection is meaningful (front hemisphere, near field)
    near = valid & (np.abs(ref["xy"][..., 0]) < 1e5) & (np.abs(ref["xy"][..., 1]) < 1e5)
    if near.any():
        assert np.abs(out["xy"] - ref["xy"])[near].max() < 1e-6
    return int(bad.sum())


CASES = {
    # name: (base config, scale overrides, focused?)
    "tiny": ("tiny", dict(), False),
    "tiny_focused": ("tiny", dict(n_orbits=3000), True),
    "mba_focused": ("small_mba", dict(n_orbits=6011, n_exp=75, width=512, height=384), True),
    "lsst_focused": ("lsst", dict(n_orbits=4100, n_exp=70, width=640, height=512), True),
    "neo_focused": ("neo", dict(n_orbits=6100, n_exp=100, width=512, height=512), True),
    "tno_focused": ("tno", dict(n_orbits=4000, n_exp=90, width=512, height=512), True),
    "neo_diffuse": ("neo", dict(n_orbits=5000, n_exp=64, width=512, height=512), False),
}


def _scene(case):
    base, kw, foc = CASES[case]
    cfg = ds.CONFIGS[base]
    if kw:
        cfg = ds.scaled(cfg, **kw)
    if foc:
        cfg = ds.focused(cfg)
    return ds.build_scene(cfg, oracle.scene_project_fn)


@pytest.mark.parametrize("flags", [4, 6], ids=["warm", "cold"])
@pytest.mark.parametrize("case", ["tiny_focused", "neo_focused"])
def test_project_parity(case, flags):
    """Steps 1-8 pair by pair against the oracle, every pair refined (dt_project's default), with the
    warm-started Kepler chain and with the cold solve."""
    dt = _dt()
    sc = _scene(case)
    el = sc.elements()[:2500]
    ref = oracle.project(oracle.Survey.from_scene(sc), el, sc.t0)
    with dt.Tracker.from_scene(sc, flags=flags) as trk:
        out = trk.project(el, sc.t0)
    n_band = _compare_project(out, ref)
    parity_record("project[%s,flags=%d]" % (case, flags), pairs=int(ref["flag"].size),
                  flagged_pairs=int(ref["flag"].sum()), in_band_pixel_mismatches=n_band)


@pytest.mark.parametrize("flags", [8, 10], ids=["warm+precull", "cold+precull"])
@pytest.mark.parametrize("case", ["tiny_focused", "neo_focused", "neo_diffuse", "tno_focused", "mba_focused"])
def test_project_precull_against_oracle(case, flags):
    """The path the timed kernel takes -- conservative cone pre-cull on a cull-quality (unpolished,
    seed-reciprocal, no-refresh) Kepler chain, precision deferred to the survivors -- compared with the
    ORACLE pair by pair (DT_FLAG_PROJECT_PRECULL makes dt_project run kernel 1 exactly as dt_stack does
    and report the pairs it culls as NaN / (-1,-1)):
      (i)  no pair the oracle marks as a hit is culled (conservativeness, against the oracle);
      (ii) every pair that survives the cull carries the oracle's sky position (1e-10 rad), pixel
           coordinates (1e-6 px) and pixel indices (exact off the guard band), i.e. the deferred polish
           restores full precision."""
    dt = _dt()
    sc = _scene(case)
    el = sc.elements()[:3000]
    ref = oracle.project(oracle.Survey.from_scene(sc), el, sc.t0)
    with dt.Tracker.from_scene(sc, flags=flags) as trk:
        out = trk.project(el, sc.t0)
    refined = np.isfinite(out["radec"][..., 0])
    ohit = ref["pix"][..., 0] >= 0
    # (i) conservativeness: an oracle hit outside the guard band must have survived and carry the same pixel
    assert not (ohit & ~refined & (ref["flag"] == 0)).any(), np.argwhere(ohit & ~refined)[:5]
    assert not (ohit & ~refined).any(), "a flagged oracle hit was culled (the cone has 1e-4 rad of slack)"
    # culled pairs report (-1, -1)
    assert (out["pix"][~refined] == -1).all()
    # (ii) survivors at full precision
    sub = dict(radec=np.where(refined[..., None], out["radec"], ref["radec"]),
               xy=np.where(refined[..., None], out["xy"], ref["xy"]),
               pix=np.where(refined[..., None], out["pix"], ref["pix"]))
    n_band = _compare_project(sub, ref)
    frac = float(refined.mean())
    if case == "neo_diffuse":           # a blind search: most warps must have been culled, else the test is vacuous
        assert frac < 0.5, "the pre-cull culled (almost) nothing"
    assert int((ohit & refined).sum()) == int(ohit.sum())
    if case != "neo_diffuse":           # a blind search of 3000 orbits hits nothing
        assert int(ohit.sum()) > 0
    parity_record("project_precull[%s,flags=%d]" % (case, flags), pairs=int(refined.size),
                  refined_fraction=frac, oracle_hits=int(ohit.sum()), flagged_pairs=int(ref["flag"].sum()),
                  in_band_pixel_mismatches=n_band)


@pytest.mark.parametrize("case", list(CASES))
def test_stack_parity(case):
    dt = _dt()
    sc = _scene(case)
    mode = sc.cfg.variance_mode
    el = sc.elements()
    flux, var = _planes(sc, mode)
    ref = oracle.stack(oracle.Survey.from_scene(sc), list(flux), list(var) if var is not None else None,
                       el, sc.t0)
    results = {}
    for flags in (0, 6):
        with dt.Tracker.from_scene(sc, flags=flags) as trk:
            trk.load_image_batch(0, flux, var)
            snr, hits = trk.stack(el, sc.t0)
            st = trk.stats()
            rep = _compare_stack(snr, hits, ref, "%s flags=%d" % (case, flags))
            assert st["pairs"] == el.shape[0] * sc.cfg.n_exp
            if rep["flagged_orbits"] == 0:
                assert st["hits"] == int(ref["hits"][ref["hits"] > 0].sum())
            results[flags] = (snr, hits)
            print(case, "flags", flags, rep, {k: st[k] for k in ("hits", "refined_pairs", "cold_solves")})
    # the fast path and the reference mode of kernel 1 agree with each other as well
    assert np.array_equal(results[0][1], results[6][1]) or ref["nflag"].any()
    if "focused" in case:
        assert ref["hits"].max() >= 2
    # top-k on the device equals the oracle's full sort of the oracle's own result (where SNR ties
    # are exact: compare indices only when the two SNR arrays agree bit for bit)
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux, var)
        snr, hits = trk.stack(el, sc.t0)
        for k, mh in [(10, 1), (257, 0), (el.shape[0] + 5, 2)]:
            idx, val = trk.topk(k, mh)
            widx, wval = oracle.topk(snr, hits, k, mh)       # oracle sort of the SAME array
            assert np.array_equal(idx, widx) and np.array_equal(val, wval)


def test_injected_source_recovered_tiny():
    """CFG 1: the injected 0.5 sigma source at node 5105 stacks to ~ A sqrt(N) and tops the list."""
    dt = _dt()
    sc = _scene("tiny")
    flux, var = _planes(sc, 1)
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux, var)
        snr, hits = trk.stack(sc.elements(), sc.t0)
        idx, val = trk.topk(5, min_hits=32)
    assert hits[5105] == 64 and abs(snr[5105] - 0.5 * 8.0) < 4.0
    assert idx[0] == 5105 and val[0] == snr[5105]


def test_address_images_exact_pixels():
    """flux = pixel address (exact in fp32), var = 1: S is the sum of addresses, so any wrong pixel
    shows up exactly; hits must equal the oracle's pixel list."""
    dt = _dt()
    sc = _scene("mba_focused")
    N, H, W = sc.cfg.n_exp, sc.cfg.height, sc.cfg.width
    el = sc.elements()
    addr = np.arange(H * W, dtype=np.float32).reshape(1, H, W).repeat(N, 0)
    sv = oracle.Survey.from_scene(sc)
    sv1 = oracle.Survey(sc.t, sc.obs_ecl, sc.ra0, sc.dec0, W, H, sc.pixel_scale, sc.gm, sc.c,
                        sc.obliquity, 0, np.ones(N))
    ref = oracle.stack(sv1, list(addr), None, el, sc.t0)
    with dt.Tracker.from_scene(sc, variance_mode=0, var_scalar=np.ones(N)) as trk:
        trk.load_image_batch(0, addr)
        snr, hits = trk.stack(el, sc.t0)
    clean = ref["nflag"] == 0
    assert np.array_equal(hits[clean], ref["hits"][clean])
    S_gpu = snr * np.sqrt(np.maximum(hits, 1))
    assert np.allclose(S_gpu[clean], ref["S"][clean], rtol=1e-12, atol=0)
    del sv


def test_masked_pixels_invalid_orbits_and_edges():
    dt = _dt()
    sc = _scene("tiny_focused")
    N, H, W = sc.cfg.n_exp, sc.cfg.height, sc.cfg.width
    el = sc.elements()[:700].copy()
    flux = np.ones((N, H, W), np.float32)
    var = np.ones((N, H, W), np.float32)
    sv = oracle.Survey.from_scene(sc)
    pix = oracle.project(sv, el, sc.t0)["pix"]
    o = 4 + int(np.argmax((pix[4:, :, 0] >= 0).sum(1)))          # not one of the orbits made invalid
    js = np.flatnonzero(pix[o, :, 0] >= 0)
    flux[js[0], pix[o, js[0], 1], pix[o, js[0], 0]] = np.nan
    var[js[1], pix[o, js[1], 1], pix[o, js[1], 0]] = 0.0
    var[js[2], pix[o, js[2], 1], pix[o, js[2], 0]] = np.inf
    el[0, 0], el[1, 1], el[2, 1], el[3, 5] = -1.0, 1.0, -0.1, np.nan
    ref = oracle.stack(sv, list(flux), list(var), el, sc.t0)
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux, var)
        snr, hits = trk.stack(el, sc.t0)
        assert trk.stats()["invalid_orbits"] == 4
        rep = _compare_stack(snr, hits, ref)
        assert list(hits[:4]) == [-1] * 4 and np.isnan(snr[:4]).all()
        # empty and single-orbit calls
        s0, h0 = trk.stack(np.zeros((0, 6)), sc.t0)
        assert s0.size == 0 and h0.size == 0
        idx, val = trk.topk(3)
        assert idx.size == 0
        s1, h1 = trk.stack(el[o:o + 1], sc.t0)
        assert h1[0] == ref["hits"][o] and abs(s1[0] - ref["snr"][o]) <= 1e-9 * abs(ref["snr"][o])
    print(rep)


def test_errors_and_state():
    dt = _dt()
    sc = _scene("tiny_focused")
    N, H, W = sc.cfg.n_exp, sc.cfg.height, sc.cfg.width
    with dt.Tracker.from_scene(sc) as trk:
        with pytest.raises(dt.DtError) as e:
            trk.stack(sc.elements()[:10], 0.0)
        assert e.value.code == dt.DT_ERR_NOT_LOADED
        with pytest.raises(dt.DtError) as e:
            trk.topk(3)
        assert e.value.code == dt.DT_ERR_STATE
        with pytest.raises(dt.DtError) as e:
            trk.load_image_batch(N - 1, np.zeros((2, H, W), np.float32), np.zeros((2, H, W), np.float32))
        assert e.value.code == dt.DT_ERR_INVALID_ARG
        with pytest.raises(dt.DtError):
            trk.load_image_batch(0, np.zeros((1, H, W), np.float32))      # mode 1 needs var
    with pytest.raises(dt.DtError):
        dt.dt_create(sc.t, sc.obs_ecl, sc.ra0, sc.dec0, 0, 16, sc.pixel_scale, var_scalar=sc.var_scalar)


def test_streaming_batches_match_resident():
    """north_star subsystem 4: a survey larger than the HBM budget is streamed from pinned host
    memory in double-buffered exposure batches; results must equal the resident run bit for bit.
    (The zero-copy gather, which would skip the copies on this short hit list, is switched off here
    and tested in test_streaming_zero_copy_gather_matches_copied_batches.)"""
    dt = _dt()
    sc = _scene("lsst_focused")
    el = sc.elements()
    flux, var = _planes(sc, 1)
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux, var)
        snr_r, hits_r = trk.stack(el, sc.t0)
        assert trk.stats()["streamed"] == 0
    pf, pv = torch.from_numpy(flux).pin_memory(), torch.from_numpy(var).pin_memory()
    per_exp = flux[0].nbytes * 2
    for nb in (9, 33):           # 9 exposures per batch (ragged, < one group) and 32 (33 rounded down)
        with dt.Tracker.from_scene(sc, hbm_budget_bytes=2 * nb * per_exp) as trk:
            with pytest.raises(dt.DtError):
                trk.load_image_batch(0, flux, var)                        # pageable: refused
            half = sc.cfg.n_exp // 2
            trk.load_image_batch(half, pf[half:], pv[half:])
            trk.load_image_batch(0, pf[:half], pv[:half])
            trk.set_option("stream_zero_copy", 0)
            trk.set_option("stream_tiles", 0)                             # whole planes, double-buffered
            snr_s, hits_s = trk.stack(el, sc.t0)
            st = trk.stats()
            assert st["streamed"] == 1 and st["n_image_batches"] == math.ceil(sc.cfg.n_exp / min(nb, 32))
            assert st["h2d_image_bytes"] == flux.nbytes + var.nbytes
            assert np.array_equal(hits_s, hits_r)
            assert np.array_equal(snr_s, snr_r)
            snr_s2, _ = trk.stack(el, sc.t0)                              # second pass reuses the slots
            assert np.array_equal(snr_s2, snr_r)


def test_many_exposures_and_device_pointers():
    """More than one exposure unit (> 512 exposures) with carried partial sums, CUDA-tensor inputs
    and outputs, and a torch stream."""
    dt = _dt()
    cfg = ds.focused(ds.scaled(ds.CONFIGS["tno"], n_orbits=2500, n_exp=600, width=128, height=128,
                               variance_mode=0))
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    el = sc.elements()
    flux, _ = _planes(sc, 0)
    ref = oracle.stack(oracle.Survey.from_scene(sc), list(flux), None, el, sc.t0)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        with dt.Tracker.from_scene(sc, stream=stream.cuda_stream) as trk:
            trk.load_image_batch(0, torch.from_numpy(flux).cuda())
            snr, hits = trk.stack(torch.from_numpy(el).cuda(), sc.t0)
            assert snr.is_cuda and hits.is_cuda
            rep = _compare_stack(snr.cpu().numpy(), hits.cpu().numpy(), ref)
            assert trk.stats()["n_image_batches"] == 2
    assert ref["hits"].max() > 100
    print(rep)


def test_more_than_one_orbit_unit():
    """> 2^20 orbits: two orbit units; oracle on a strided sample plus the tail."""
    dt = _dt()
    cfg = ds.focused(ds.scaled(ds.CONFIGS["small_mba"], n_orbits=(1 << 20) + 4097, n_exp=40, width=256,
                               height=256))
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    el = sc.elements()
    flux, _ = _planes(sc, 0)
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux)
        snr, hits = trk.stack(el, sc.t0)
    sel = np.concatenate([np.arange(0, el.shape[0], 37), np.arange((1 << 20) - 300, el.shape[0])])
    ref = oracle.stack(oracle.Survey.from_scene(sc), list(flux), None, el[sel], sc.t0)
    rep = _compare_stack(snr[sel], hits[sel], ref)
    assert ref["hits"].max() >= 2
    print(rep)


@pytest.mark.parametrize("var_mode", [0, 1], ids=["scalar_var", "plane_var"])
@pytest.mark.parametrize("schedule", ["auto", "orbit_major", "orbit_major_slabs", "auto_slabs", "dense"])
def test_gather_hits_entry_matches_definition(schedule, var_mode):
    """dt_gather_hits on a hand-built hit list: every pair hits a seeded random pixel.  Every schedule of
    kernel 3 (forced through dt_set_option) and the library's own choice must give exactly the sequential sums of the definition,
    with a per-exposure scalar variance and with variance planes."""
    dt = _dt()
    N, H, W, n = 64, 96, 80, 1000
    rng = np.random.default_rng(5)
    t = np.linspace(0, 10, N)
    var_s = rng.uniform(0.8, 1.2, N)
    flux = rng.normal(size=(N, H, W)).astype(np.float32)
    npad = (n + 31) // 32 * 32
    hit = rng.random((N, npad)) < 0.3
    hit[:, n:] = False
    pixel = rng.integers(0, H * W, size=(N, npad))
    G = N // 32
    mask = np.zeros((G, npad), np.uint32)
    base = np.zeros((G, npad // 32), np.uint64)
    offsets = []
    for g in range(G):
        for w in range(npad // 32):
            base[g, w] = len(offsets)
            for b in range(32):                       # exposure-ascending, then lane-ascending
                for o in range(32 * w, 32 * w + 32):
                    if hit[32 * g + b, o]:
                        mask[g, o] |= np.uint32(1 << b)
                        offsets.append((b << 27) | pixel[32 * g + b, o])   # entry = exposure tag | offset
    offsets = np.array(offsets, np.uint32)
    S = np.zeros(n)
    Wt = np.zeros(n)
    var = rng.uniform(0.5, 2.0, size=(N, H, W)).astype(np.float32) if var_mode == 1 else None
    for o in range(n):
        for j in range(N):
            if hit[j, o]:
                v = np.float64(var[j].reshape(-1)[pixel[j, o]]) if var_mode == 1 else var_s[j]
                S[o] += np.float64(flux[j].reshape(-1)[pixel[j, o]]) / v
                Wt[o] += 1.0 / v
    with dt.Tracker(t, ds.observer_ecliptic(t), np.zeros(N), np.zeros(N), W, H, ds.PIXEL_SCALE,
                    variance_mode=var_mode, var_scalar=var_s) as trk:
        trk.load_image_batch(0, flux, var)
        trk.set_option("gather_schedule", {"auto": -1, "orbit_major": 0, "orbit_major_slabs": 0, "auto_slabs": -1,
                                           "dense": 1}[schedule])
        if schedule.endswith("_slabs"):          # the walk launched once per exposure group, sums carried between them
            trk.set_option("gather_slab", 1)
        dS = torch.zeros(n, dtype=torch.float64, device="cuda")
        dW = torch.zeros(n, dtype=torch.float64, device="cuda")
        dc = torch.zeros(n, dtype=torch.int32, device="cuda")
        trk.gather_hits(n, 0, G, torch.from_numpy(mask.view(np.int32)).cuda(),
                        torch.from_numpy(base.view(np.int64)).cuda(),
                        torch.from_numpy(offsets.view(np.int32)).cuda(), len(offsets), dS, dW, dc)
        torch.cuda.synchronize()
    assert np.array_equal(dc.cpu().numpy(), hit[:, :n].sum(0).astype(np.int32))
    assert np.array_equal(dS.cpu().numpy(), S) and np.array_equal(dW.cpu().numpy(), Wt)


def test_bounds_check_build_catches_a_corrupt_hit_list():
    """compute-sanitizer is closed on the GPU pool (profiles/r2_memcheck.md); its stand-in is the -DDT_BOUNDS_CHECK
    build (python -m paper_2503_08854_b200._build --bounds; DTRACK_LIB=.../libdtrack_bounds.so pytest -m gpu): every
    data-dependent index is checked on the device.  With that build loaded, a hit list whose entry points outside the
    plane, or whose block base points outside the list, must be refused; with the normal build the test only checks
    that a well-formed list passes."""
    dt = _dt()
    N, H, W, n = 32, 64, 64, 64
    t = np.linspace(0, 5, N)
    flux = np.ones((N, H, W), np.float32)
    mask = np.zeros((1, n), np.uint32)
    mask[0, 5] = 1                                        # orbit 5 hits exposure 0
    base = np.zeros((1, n // 32), np.uint64)
    bounds = "+bounds" in dt.dt_version()
    with dt.Tracker(t, ds.observer_ecliptic(t), np.zeros(N), np.zeros(N), W, H, ds.PIXEL_SCALE, variance_mode=0,
                    var_scalar=np.ones(N)) as trk:
        trk.load_image_batch(0, flux)
        trk.set_option("gather_schedule", 0)

        def run(entry, base0=0):
            b = base.copy()
            b[0, 0] = base0
            dS = torch.zeros(n, dtype=torch.float64, device="cuda")
            dW = torch.zeros(n, dtype=torch.float64, device="cuda")
            dc = torch.zeros(n, dtype=torch.int32, device="cuda")
            trk.gather_hits(n, 0, 1, torch.from_numpy(mask.view(np.int32)).cuda(), torch.from_numpy(b.view(np.int64)).cuda(),
                            torch.tensor([entry], dtype=torch.int32).cuda(), 1, dS, dW, dc)
            torch.cuda.synchronize()
            return int(dc.sum())

        assert run(7 * W + 3) == 1
        if bounds:
            with pytest.raises(dt.DtError):
                run(H * W + 10)                           # pixel offset outside the plane
            with pytest.raises(dt.DtError):
                run(7 * W + 3, base0=1000)                # block base outside the list
    print("library:", dt.dt_version())


def test_fp64_peak_probe_runs():
    dt = _dt()
    tf = dt.dt_fp64_peak(0)
    print("FP64 DFMA peak: %.2f TFLOP/s" % tf)
    assert 5.0 < tf < 100.0


def test_pinned_elements_zero_copy_matches_device_path():
    """dt_stack with page-locked host elements (kernel 1 bulk-copies each tile straight from host
    memory and leaves the device copy for the later exposure units and the finalisation) and
    caller-supplied pinned outputs == the device-pointer path, bit for bit; several orbit tiles with a
    ragged tail, two exposure units (streaming forces more than one pass over the orbits)."""
    dt = _dt()
    sc = _scene("mba_focused")
    cfg = sc.cfg
    flux, _ = _planes(sc, 0)
    el = sc.elements()[:5003]
    el[17, 0] = -1.0                                   # an invalid orbit rides along
    n = el.shape[0]
    el_pin = torch.from_numpy(el.copy()).pin_memory()
    out = (torch.empty(n, dtype=torch.float64).pin_memory(), torch.empty(n, dtype=torch.int32).pin_memory())
    res = {}
    for mode in ("device", "pinned", "pinned_streamed"):
        kw = {}
        if mode == "pinned_streamed":
            kw = dict(flags=1, hbm_budget_bytes=2 * 40 * cfg.plane_pixels * 4)   # 40-exposure batches
        with dt.Tracker.from_scene(sc, **kw) as trk:
            if mode == "pinned_streamed":
                fp = torch.from_numpy(flux).pin_memory()
                trk.load_image_batch(0, fp)
            else:
                trk.load_image_batch(0, flux)
            if mode == "device":
                s, h = trk.stack(torch.from_numpy(el).cuda(), sc.t0)
                res[mode] = (s.cpu().numpy(), h.cpu().numpy())
            else:
                s, h = trk.stack(el_pin, sc.t0, out=out)
                assert s is out[0] and h is out[1]
                res[mode] = (s.numpy().copy(), h.numpy().copy())
                if mode == "pinned_streamed":
                    assert trk.stats()["streamed"] == 1
    for mode in ("pinned", "pinned_streamed"):
        assert np.array_equal(res[mode][1], res["device"][1])
        assert np.array_equal(res[mode][0], res["device"][0], equal_nan=True)
    assert res["device"][1][17] == -1 and np.isnan(res["device"][0][17])


@pytest.mark.parametrize("e_hi", [0.9, 0.99], ids=["e<=0.9", "e<=0.99"])
@pytest.mark.parametrize("flags", [0, 2], ids=["warm", "cold"])
def test_perihelion_stress_all_kepler_paths(flags, e_hi):
    """Eccentric orbits (e up to 0.9) whose perihelion passages fall inside the exposure span, with
    exposure gaps from minutes to weeks: the warm step at its three orders, the wide step, wide
    sub-steps and the cold solve are all taken (counted), and every sky position / pixel coordinate
    must still match the oracle (1e-10 rad; continuous pixel coordinates to 1e-6 px; pixel indices
    exact off the guard band).  Eight families of orbits, each around a guide the tangent points track in
    turn, keep an eighth of all pairs near-field."""
    dt = _dt()
    rng = np.random.default_rng(11)
    N, n, W, H = 200, 2048, 512, 512
    gaps = np.concatenate([rng.uniform(0.003, 0.05, 60), rng.uniform(0.05, 1.0, 80), rng.uniform(1.0, 20.0, 59)])
    rng.shuffle(gaps)
    t = np.concatenate([[0.0], np.cumsum(gaps)])
    G = 8                                                    # guide orbits; families of n / G members
    ga = rng.uniform(0.8, 1.6, G)
    # e_hi = 0.99: beyond the range of every config (e <= 0.9) but inside what the ABI accepts (e < 1): such orbits
    # take no cone pre-cull (orbit_setup) and must still match the oracle through every Kepler path
    ge = np.concatenate([rng.uniform(e_hi - 0.02, e_hi, G // 2), rng.uniform(0.6 if e_hi <= 0.9 else 0.91, e_hi - 0.02, G - G // 2)])
    period = 2 * np.pi / np.sqrt(ds.GM_SUN / ga ** 3)
    t_peri = rng.uniform(0.2, 0.8, G) * t[-1]                # a perihelion passage inside the span
    guides = np.stack([ga, ge, rng.uniform(0, 0.5, G), rng.uniform(0, 2 * np.pi, G), rng.uniform(0, 2 * np.pi, G),
                       -2 * np.pi / period * t_peri], 1)
    fam = np.repeat(np.arange(G), n // G)
    el = guides[fam] + rng.uniform(-1, 1, (n, 6)) * np.array([1e-5, 1e-5, 3e-5, 3e-5, 3e-5, 3e-5])
    el[::n // G] = guides                                    # member 0 of each family is the guide itself
    obs = ds.observer_ecliptic(t)
    probe = oracle.Survey(t, obs, np.zeros(N), np.zeros(N), W, H, ds.PIXEL_SCALE, ds.GM_SUN, ds.C_AU_PER_DAY,
                          ds.OBLIQUITY, 0, np.ones(N))
    gr = oracle.project(probe, guides, 0.0)["radec"]         # [G, N, 2]
    track = gr[np.arange(N) % G, np.arange(N)]               # exposure j looks at guide j mod G
    sv = oracle.Survey(t, obs, track[:, 0], track[:, 1], W, H, ds.PIXEL_SCALE, ds.GM_SUN, ds.C_AU_PER_DAY,
                       ds.OBLIQUITY, 0, np.ones(N))
    ref = oracle.project(sv, el, 0.0)
    with dt.Tracker(t, obs, track[:, 0], track[:, 1], W, H, ds.PIXEL_SCALE, variance_mode=0, var_scalar=np.ones(N),
                    flags=flags) as trk:
        out = trk.project(el, 0.0)
        n_bad = _compare_project(out, ref)
        trk.load_image_batch(0, np.ones((N, H, W), np.float32))
        snr, hits = trk.stack(el, 0.0)
        st = trk.stats()
    # the timed path (pre-cull where the orbit has one) finds exactly the oracle's hits
    want = (ref["pix"][..., 0] >= 0).sum(1)
    nfl = ref["flag"].astype(np.int64).sum(1)
    assert np.array_equal(hits[nfl == 0], want[nfl == 0]) and (np.abs(hits - want) <= nfl).all()
    # a guide is seen in every exposure that tracks it; unit images: SNR = sqrt(hits)
    assert hits[0] >= N // G and abs(snr[0] - math.sqrt(hits[0])) < 1e-12
    near = (np.abs(ref["xy"]) < 1e5).all(-1)
    assert near.sum() > 0.1 * n * N                          # the 1e-6 px comparison covered many pairs
    if flags == 0:
        assert st["substep_solves"] > 0.05 * n * N, st          # wide steps / sub-steps were exercised
        assert 0 < st["cold_solves"] < 0.5 * n * N, st          # and so was the cold solve, but rarely
    print("perihelion stress: flagged pixel mismatches %d, substep %d, cold %d of %d pairs" %
          (n_bad, st["substep_solves"], st["cold_solves"], n * N))


@pytest.mark.parametrize("case,expect_auto", [("neo_diffuse", 1), ("tno_focused", None)])
def test_streaming_zero_copy_gather_matches_copied_batches(case, expect_auto):
    """Streaming mode has two ways to reach the pixels: copy every exposure batch into the double
    buffer, or -- when a probe predicts few hits -- gather straight from the page-locked host planes.
    Forced copy, forced zero-copy and the library's own choice must agree bit for bit with each other
    and with the resident run; the choice is zero-copy on a blind (diffuse) list."""
    dt = _dt()
    sc = _scene(case)
    cfg = sc.cfg
    el = sc.elements()
    flux, var = _planes(sc, cfg.variance_mode)
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux, var)
        snr_r, hits_r = trk.stack(el, sc.t0)
    pf = torch.from_numpy(flux).pin_memory()
    pv = torch.from_numpy(var).pin_memory() if var is not None else None
    per_exp = flux[0].nbytes * (2 if var is not None else 1)
    for mode, want in ((0, 0), (1, 1), (-1, expect_auto)):
        with dt.Tracker.from_scene(sc, hbm_budget_bytes=2 * 20 * per_exp) as trk:
            trk.set_option("stream_zero_copy", mode)
            trk.set_option("stream_tiles", 0)                             # the tile cache has its own test
            trk.load_image_batch(0, pf, pv)
            snr_s, hits_s = trk.stack(el, sc.t0)
            st = trk.stats()
        assert st["streamed"] == 1
        if want is not None:
            assert st["image_zero_copy"] == want, (mode, st)
        assert (st["h2d_image_bytes"] == 0) == (st["image_zero_copy"] == 1)
        assert np.array_equal(hits_s, hits_r) and np.array_equal(snr_s, snr_r), mode


@pytest.mark.parametrize("case", ["lsst_focused", "tno_focused", "mba_focused"])
def test_streaming_tile_cache_matches_resident(case):
    """hits first, then only the 64 x 64-pixel tiles the hits fall on cross PCIe into a device
    tile cache; pixels of tiles without a slot are read zero-copy.  Bit-identical to the resident run with the
    default fetch threshold, with every touched tile fetched, with a cache of five slots (overflow -> zero-copy),
    and with a 3 x 3 patch that crosses tile borders; fewer bytes move than the planes hold."""
    dt = _dt()
    sc = _scene(case)
    cfg = sc.cfg
    el = sc.elements()
    flux, var = _planes(sc, cfg.variance_mode)
    w3 = np.array([[0.1, 0.2, 0.1], [0.2, 1.0, 0.2], [0.1, 0.2, 0.1]])
    with dt.Tracker.from_scene(sc) as trk:
        trk.load_image_batch(0, flux, var)
        snr_r, hits_r = trk.stack(el, sc.t0)
        trk.set_patch(3, w3)
        snr_p, hits_p = trk.stack(el, sc.t0)
    pf = torch.from_numpy(flux).pin_memory()
    pv = torch.from_numpy(var).pin_memory() if var is not None else None
    planes = 2 if var is not None else 1
    per_exp = flux[0].nbytes * planes
    slot_bytes = 64 * 64 * 4 * planes
    full = flux.nbytes * planes
    fetched = {}
    for label, budget, min_hits, patch in [("default", 20 * per_exp, 0, 1), ("all_tiles", 20 * per_exp, 1, 1),
                                           ("five_slots", 5 * slot_bytes, 1, 1), ("patch3", 20 * per_exp, 4, 3)]:
        with dt.Tracker.from_scene(sc, hbm_budget_bytes=budget) as trk:
            trk.set_option("stream_zero_copy", 0)                         # not the pure zero-copy gather
            trk.set_option("tile_min_hits", min_hits)
            trk.load_image_batch(0, pf, pv)
            if patch > 1:
                trk.set_patch(3, w3)
            snr_s, hits_s = trk.stack(el, sc.t0)
            st = trk.stats()
            snr_s2, _ = trk.stack(el, sc.t0)                              # the cache is rebuilt per call
        assert st["streamed"] == 1 and st["image_tiles"] == 1 and st["image_zero_copy"] == 0, (label, st)
        assert st["h2d_image_bytes"] == st["tiles_fetched"] * slot_bytes
        want = (snr_p, hits_p) if patch > 1 else (snr_r, hits_r)
        assert np.array_equal(hits_s, want[1]) and np.array_equal(snr_s, want[0]), label
        assert np.array_equal(snr_s2, want[0]), label
        fetched[label] = st["tiles_fetched"]
    assert fetched["all_tiles"] > 0 and fetched["all_tiles"] >= fetched["default"]
    assert fetched["five_slots"] <= 5 * ((cfg.n_exp + 511) // 512)        # the cache holds five tiles per exposure unit
    assert fetched["all_tiles"] * slot_bytes < full, "the tile cache must move fewer bytes than the planes hold"
    parity_record("tile_cache[%s]" % case, tiles_fetched=fetched, tile_bytes=slot_bytes, plane_bytes_total=int(full))


@pytest.mark.parametrize("case", ["neo", "small_mba", "tno", "neo+focused", "small_mba+focused", "tno+focused"])
def test_precull_is_conservative_at_scale(case):
    """The pre-cull (cone test on the geometric, possibly unpolished, position) may only drop pairs
    that cannot hit: dt_stack with and without it (DT_FLAG_NO_PRECULL refines every pair at full
    precision) must give identical hit counts and SNR for every orbit -- checked on 2e5 orbits x all
    exposures of the config's survey geometry with small planes (1e8 pairs; eccentric NEOs at all
    distances included), where any wrongly culled pair would show up."""
    dt = _dt()
    base = case.split("+")[0]
    cfg = ds.scaled(ds.CONFIGS[base], n_orbits=200_000, n_exp=min(ds.CONFIGS[base].n_exp, 500))
    if case.endswith("+focused"):       # thousands of hits per exposure, many of them near the footprint edge
        cfg = ds.focused(cfg)
    sc = ds.build_scene(cfg, oracle.scene_project_fn if case.endswith("+focused") else None, inject=False)
    el = torch.from_numpy(sc.elements()).cuda()
    g = torch.Generator(device="cuda")
    g.manual_seed(3)
    # one shared random plane stands in for all exposures (pixel values only matter for equality)
    plane = torch.randn((1, cfg.height, cfg.width), generator=g, device="cuda", dtype=torch.float32)
    vplane = torch.full_like(plane, 1.25) if cfg.variance_mode == 1 else None
    out = {}
    for flags in (0, 4):
        with dt.Tracker.from_scene(sc, flags=flags, hbm_budget_bytes=cfg.image_bytes() + (1 << 30)) as trk:
            for j in range(cfg.n_exp):
                trk.load_image_batch(j, plane, vplane)
            snr, hits = trk.stack(el, sc.t0)
            st = trk.stats()
            out[flags] = (snr.cpu().numpy(), hits.cpu().numpy(), st["hits"], st["refined_pairs"])
    assert out[0][2] == out[4][2] and out[0][2] > 0, (out[0][2], out[4][2])
    assert np.array_equal(out[0][1], out[4][1])
    assert np.array_equal(out[0][0], out[4][0])
    if not case.endswith("+focused"):
        assert out[0][3] < 0.05 * out[4][3]      # and it does cull
    print(case, "hits", out[0][2], "refined pairs with / without the pre-cull", out[0][3], out[4][3])


# ---- group ephemeris gate (reading A25) ----------------------------------------------------------------------
GATE_CASES = {
    # full cadence (the gate's remainder bound grows with the cube of a group's half-span, so the reduced
    # exposure counts of CASES would switch it off), reduced planes and orbit counts; (base, overrides, guides)
    "mba": ("small_mba", dict(n_orbits=4096, width=512, height=384), 24),
    "lsst": ("lsst", dict(n_orbits=3072, n_exp=1200, width=320, height=256), 24),
    "neo": ("neo", dict(n_orbits=4096, width=512, height=512), 24),
    "tno": ("tno", dict(n_orbits=3072, width=320, height=320), 4),
}


def _gate_scene(case):
    """A focused search whose orbits are re-ordered so that every warp tile of 32 holds members of ONE family (then
    the diffuse orbits): at the exposures that follow another guide all 32 lanes are far and the gate decides for the
    whole warp; at the exposures of the tile's own guide all 32 sit inside or at the edge of the footprint at once."""
    base, kw, n_guides = GATE_CASES[case]
    cfg = ds.focused(ds.scaled(ds.CONFIGS[base], **kw), n_guides=n_guides)
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    el = sc.elements()
    guides = ds.workloads.guide_elements(cfg)
    d = np.abs(el[:, None, :] - guides[None, :, :]).max(-1)
    fam, member = d.argmin(-1), d.min(-1) < 0.05
    order = np.concatenate([np.flatnonzero(member & (fam == g)) for g in range(guides.shape[0])] +
                           [np.flatnonzero(~member)])
    return sc, np.ascontiguousarray(el[order])


@pytest.mark.parametrize("case", list(GATE_CASES))
def test_group_gate_against_oracle(case):
    """The gate must never remove a pair the oracle reports as a hit, whatever it does to the others, and the pairs
    that reach the per-pair path keep full precision (dt_project under DT_FLAG_PROJECT_PRECULL = kernel 1 exactly
    as dt_stack runs it, gate included; flags 24 = the same without the gate)."""
    dt = _dt()
    sc, el = _gate_scene(case)
    el = el[:2048]
    ref = oracle.project(oracle.Survey.from_scene(sc), el, sc.t0)
    ohit = ref["pix"][..., 0] >= 0
    fr = {}
    for flags in (8, 24):
        with dt.Tracker.from_scene(sc, flags=flags) as trk:
            out = trk.project(el, sc.t0)
        refined = np.isfinite(out["radec"][..., 0])
        assert not (ohit & ~refined).any(), (flags, np.argwhere(ohit & ~refined)[:5])
        assert (out["pix"][~refined] == -1).all()
        sub = dict(radec=np.where(refined[..., None], out["radec"], ref["radec"]),
                   xy=np.where(refined[..., None], out["xy"], ref["xy"]),
                   pix=np.where(refined[..., None], out["pix"], ref["pix"]))
        _compare_project(sub, ref)
        fr[flags] = float(refined.mean())
    assert int(ohit.sum()) > 100, "no hits: the test would be vacuous"
    assert fr[8] <= fr[24] + 1e-12
    parity_record("group_gate_project[%s]" % case, pairs=int(ohit.size), oracle_hits=int(ohit.sum()),
                  refined_fraction_gate=fr[8], refined_fraction_no_gate=fr[24])


@pytest.mark.parametrize("case", list(GATE_CASES))
def test_group_gate_changes_nothing(case):
    """dt_stack with the gate forced on, switched off, and chosen on the device: SNR and hit counts are bit-identical
    (the gate only removes pairs that are no hits), and where its bounds are tight it really removes most of the
    per-pair Kepler steps of these searches."""
    dt = _dt()
    sc, el = _gate_scene(case)
    flux, var = _planes(sc, sc.cfg.variance_mode)
    res = {}
    for gate in (1, 0, -1):
        with dt.Tracker.from_scene(sc) as trk:
            trk.set_option("group_gate", gate)
            trk.load_image_batch(0, flux, var)
            snr, hits = trk.stack(el, sc.t0)
            res[gate] = (np.array(snr), np.array(hits), trk.stats())
    for gate in (0, -1):
        assert np.array_equal(res[1][1], res[gate][1])
        assert np.array_equal(res[1][0], res[gate][0], equal_nan=True)
        assert res[1][2]["hits"] == res[gate][2]["hits"]
    st = res[1][2]
    assert res[0][2]["gated_pairs"] == 0 and st["hits"] > 100
    frac = st["gated_pairs"] / st["pairs"]
    if case != "neo":                      # eccentric near-Earth orbits: the bounds are loose next to a perihelion
        assert frac > 0.5, frac
    parity_record("group_gate_stack[%s]" % case, pairs=int(st["pairs"]), hits=int(st["hits"]),
                  gated_fraction=frac, gated_fraction_device_choice=res[-1][2]["gated_pairs"] / st["pairs"],
                  refined_fraction=st["refined_pairs"] / st["pairs"],
                  refined_fraction_no_gate=res[0][2]["refined_pairs"] / res[0][2]["pairs"])


def test_group_gate_device_choice():
    """The device-side policy: a blind search (every warp culls) keeps the gate from unit to unit; a focused search
    whose family members are scattered over the warps (most pairs refined) drops it after its first unit -- unless
    the orbits are put into sky order first (the default), which makes the warps of such a search homogeneous and
    lets the gate work there too.  Results equal the gate-less run."""
    dt = _dt()
    out = {}
    for name, foc, sort in (("blind", False, 1), ("focused_caller_order", True, 0), ("focused_sky_order", True, 1)):
        cfg = ds.scaled(ds.CONFIGS["lsst"], n_orbits=8192, width=160, height=128)       # 2000 exposures: 4 units
        if foc:
            cfg = ds.focused(cfg)
        sc = ds.build_scene(cfg, oracle.scene_project_fn)
        flux, var = _planes(sc, cfg.variance_mode)
        el = sc.elements()
        runs = {}
        for flags in (0, 16):
            with dt.Tracker.from_scene(sc, flags=flags) as trk:
                trk.set_option("sort_orbits", sort)
                trk.load_image_batch(0, flux, var)
                snr, hits = trk.stack(el, sc.t0)
                runs[flags] = (np.array(snr), np.array(hits), trk.stats())
        assert np.array_equal(runs[0][1], runs[16][1]) and np.array_equal(runs[0][0], runs[16][0], equal_nan=True)
        st = runs[0][2]
        out[name] = st["gated_pairs"] / st["pairs"]
        assert st["launches"] == 3 * st["propagate_launches"] + st["gather_launches"] + 1
    assert out["blind"] > 0.8, out                      # all four units gated
    assert out["focused_caller_order"] < 0.3, out       # at most the first of four units ran the gate variant
    assert out["focused_sky_order"] > 0.5, out
    parity_record("group_gate_device_choice", gated_fraction=out)


@pytest.mark.parametrize("case", ["tiny_focused", "mba_focused", "neo_focused", "tno_focused", "neo_diffuse"])
def test_sky_order_changes_nothing_but_rounding(case):
    """dt_stack in sky order (the default) and in the caller's order: both against the oracle, and against each other
    -- the same hit counts wherever the oracle flags no pair, SNR to 1e-9 (not bit for bit: which Kepler series a warp
    takes is a warp vote, and the warps differ).  Per-orbit epochs travel with their orbits."""
    dt = _dt()
    sc = _scene(case)
    el = sc.elements()
    flux, var = _planes(sc, sc.cfg.variance_mode)
    ref = oracle.stack(oracle.Survey.from_scene(sc), list(flux), list(var) if var is not None else None, el, sc.t0)
    res = {}
    for sort in (1, 0):
        with dt.Tracker.from_scene(sc) as trk:
            trk.set_option("sort_orbits", sort)
            trk.load_image_batch(0, flux, var)
            snr, hits = trk.stack(el, sc.t0)
            _compare_stack(snr, hits, ref, "%s sort=%d" % (case, sort))
            res[sort] = (np.array(snr), np.array(hits))
            if sort == 1:
                # per-orbit epochs, shifted by whole periods' worth of mean anomaly: M0' = M0 + n dt at t0 + dt
                rs = np.random.RandomState(3)
                dtv = rs.uniform(-50.0, 50.0, el.shape[0])
                n_mot = np.sqrt(sc.gm / el[:, 0] ** 3) if hasattr(sc, "gm") else None
                if n_mot is not None:
                    el2 = el.copy()
                    el2[:, 5] = el[:, 5] + n_mot * dtv
                    snr2, hits2 = trk.stack(el2, sc.t0 + dtv)
                    clean = ref["nflag"] == 0
                    assert np.array_equal(np.asarray(hits2)[clean], ref["hits"][clean])
    clean = ref["nflag"] == 0
    assert np.array_equal(res[0][1][clean], res[1][1][clean])
    same = clean & (res[0][1] == res[1][1])
    a, b = res[0][0][same], res[1][0][same]
    ok = (np.isnan(a) & np.isnan(b)) | (np.abs(a - b) <= 1e-9 * np.maximum(np.abs(b), 1e-3))
    assert ok.all()


def test_group_level_gate_against_oracle():
    """The group-level test of the gate (one bounding-cone test per orbit and group where a group's pointings cluster:
    dt_orbit.cuh group_is_far) on the survey geometry that switches it on -- pointings that follow the opposition
    point, configs[1] at full cadence -- with pixels 100 times coarser than the configs', so that a blind set of
    main-belt orbits has over a thousand oracle hits to lose: none may be removed, survivors keep full precision, and the
    test must really remove most (orbit, group) pairs."""
    dt = _dt()
    cfg = ds.scaled(ds.CONFIGS["small_mba"], n_orbits=8192, width=512, height=384)
    sc = ds.build_scene(cfg, oracle.scene_project_fn, inject=False)
    scale = 100.0 * sc.pixel_scale                         # 20 arcsec per pixel: a 2.8 x 2.1 degree footprint
    el = sc.elements()
    srv = oracle.Survey(sc.t, sc.obs_ecl, sc.ra0, sc.dec0, cfg.width, cfg.height, scale, sc.gm, sc.c, sc.obliquity)
    ref = oracle.project(srv, el, sc.t0)
    ohit = ref["pix"][..., 0] >= 0
    assert int(ohit.sum()) > 1000, int(ohit.sum())
    fr = {}
    for flags in (8, 24):
        with dt.Tracker(sc.t, sc.obs_ecl, sc.ra0, sc.dec0, cfg.width, cfg.height, scale, gm=sc.gm, c=sc.c,
                        obliquity=sc.obliquity, variance_mode=0, var_scalar=np.ones(cfg.n_exp), flags=flags) as trk:
            out = trk.project(el, sc.t0)
        refined = np.isfinite(out["radec"][..., 0])
        assert not (ohit & ~refined).any(), (flags, np.argwhere(ohit & ~refined)[:5])
        assert (out["pix"][~refined] == -1).all()
        sub = dict(radec=np.where(refined[..., None], out["radec"], ref["radec"]),
                   xy=np.where(refined[..., None], out["xy"], ref["xy"]),
                   pix=np.where(refined[..., None], out["pix"], ref["pix"]))
        _compare_project(sub, ref)
        fr[flags] = float(refined.mean())
    assert fr[8] <= fr[24] + 1e-12
    # dt_stack statistics on the same geometry: most pairs gated, same hits with and without
    flux = np.zeros((cfg.n_exp, cfg.height, cfg.width), np.float32)
    st = {}
    for gate in (1, 0):
        with dt.Tracker(sc.t, sc.obs_ecl, sc.ra0, sc.dec0, cfg.width, cfg.height, scale, gm=sc.gm, c=sc.c,
                        obliquity=sc.obliquity, variance_mode=0, var_scalar=np.ones(cfg.n_exp)) as trk:
            trk.set_option("group_gate", gate)
            trk.load_image_batch(0, flux, None)
            snr, hits = trk.stack(el, sc.t0)
            st[gate] = (np.array(hits), trk.stats())
    assert np.array_equal(st[1][0], st[0][0])
    clean = ref["flag"].sum(-1) == 0
    assert np.array_equal(st[1][0][clean], ohit.sum(-1)[clean])
    assert st[1][1]["gated_pairs"] > 0.6 * st[1][1]["pairs"], st[1][1]
    parity_record("group_level_gate", pairs=int(ohit.size), oracle_hits=int(ohit.sum()),
                  refined_fraction_gate=fr[8], refined_fraction_no_gate=fr[24],
                  gated_fraction=st[1][1]["gated_pairs"] / st[1][1]["pairs"])
