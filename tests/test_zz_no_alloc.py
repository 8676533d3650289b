"""dt_threshold_noalloc (include/dtrack.h): threshold mode with its scratch in a static device array -- for
callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops).  Compared with the existing
path, dt_threshold, on the same dt_stack result, twice in a row (the static array keeps the last call's
contents), bit for bit: indices are integers and the SNR values are copies.

Collected last on purpose (the suite runs with `pytest -x`).  The test passes alone in a fresh process and
after the other GPU tests: it depends on nothing but its own context."""
import numpy as np
import pytest

import dtsynth as ds
import oracle

pytestmark = pytest.mark.gpu


def _dt():
    import paper_2503_08854_b200 as dt
    return dt


def _stacked(dt, torch):
    cfg = ds.focused(ds.scaled(ds.CONFIGS["tiny"], n_orbits=3000))
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    N = cfg.n_exp
    flux = np.stack([sc.flux_plane_np(j) for j in range(N)])
    var = np.stack([sc.var_plane_np(j) for j in range(N)])
    trk = dt.Tracker.from_scene(sc)
    trk.load_image_batch(0, flux, var)
    el = torch.from_numpy(sc.elements()).cuda()
    snr, hits = trk.stack(el, sc.t0)                 # DT_MEM_DEVICE outputs: torch CUDA tensors
    return trk, snr, hits


def test_threshold_noalloc_matches_dt_threshold_twice():
    import torch
    dt = _dt()
    trk, snr, hits = _stacked(dt, torch)
    try:
        n = snr.numel()
        assert int((hits > 0).sum()) > 100
        idx = torch.empty(n, dtype=torch.int64, device="cuda")
        val = torch.empty(n, dtype=torch.float64, device="cuda")
        nf = torch.zeros(1, dtype=torch.int64, device="cuda")
        dt.dt_threshold_noalloc(snr, hits, 0.0, 0, idx, val, nf)      # loads the kernels (CUDA loads modules lazily)
        torch.cuda.synchronize()
        # first a permissive threshold (many results), then a strict one (few): stale candidates of the first
        # call must not leak into the second; then a truncated output (max_out < found)
        for snr_min, min_hits, max_out in [(-1.0, 1, n), (1.5, 8, n), (0.0, 1, 7)]:
            want_idx, want_val, want_n = trk.threshold(snr_min, min_hits, max_out)        # the existing path
            idx.fill_(-7)
            val.fill_(-7.0)
            free_before = torch.cuda.mem_get_info()[0]
            dt.dt_threshold_noalloc(snr, hits, snr_min, min_hits, idx[:max_out], val[:max_out], nf)
            torch.cuda.synchronize()
            assert torch.cuda.mem_get_info()[0] == free_before        # the device's free memory did not move
            got_n = int(nf.item())
            assert got_n == want_n and want_n > 0
            m = min(got_n, max_out)
            assert np.array_equal(idx[:m].cpu().numpy(), want_idx)
            assert np.array_equal(val[:m].cpu().numpy(), want_val)
            assert (idx[m:] == -7).all() and (val[m:] == -7.0).all()                      # nothing written beyond m
        # without the SNR output, on a side stream
        st = torch.cuda.Stream()
        st.wait_stream(torch.cuda.current_stream())
        want_idx, _, want_n = trk.threshold(0.5, 2, n)
        dt.dt_threshold_noalloc(snr, hits, 0.5, 2, idx, None, nf, stream=st)
        st.synchronize()
        assert int(nf.item()) == want_n and np.array_equal(idx[:want_n].cpu().numpy(), want_idx)
    finally:
        trk.close()


def test_threshold_noalloc_limits():
    import torch
    dt = _dt()
    n = dt.DT_NOALLOC_MAX_ORBITS
    g = torch.Generator(device="cuda").manual_seed(5)
    snr = torch.randn(n + 1, dtype=torch.float64, device="cuda", generator=g)
    snr[::1001] = float("nan")
    hits = torch.randint(0, 5, (n + 1,), dtype=torch.int32, device="cuda", generator=g)
    idx = torch.empty(n + 1, dtype=torch.int64, device="cuda")
    val = torch.empty(n + 1, dtype=torch.float64, device="cuda")
    nf = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    with pytest.raises(dt.DtError) as ei:                       # one more than the static array is built for
        dt.dt_threshold_noalloc(snr, hits, 0.0, 0, idx, val, nf)
    assert ei.value.code == -6 and "DT_NOALLOC_MAX_ORBITS" in str(ei.value)
    assert int(nf.item()) == -1                                 # nothing was enqueued
    # exactly the maximum, against numpy's definition; then the empty array (count cleared, nothing else touched)
    for rep in range(2):
        dt.dt_threshold_noalloc(snr[:n], hits[:n], 1.0, 2, idx[:n], val[:n], nf)
        torch.cuda.synchronize()
        s, h = snr[:n].cpu().numpy(), hits[:n].cpu().numpy()
        want = np.flatnonzero(np.isfinite(s) & (s >= 1.0) & (h >= 2))
        m = int(nf.item())
        assert m == want.size and np.array_equal(idx[:m].cpu().numpy(), want)
        assert np.array_equal(val[:m].cpu().numpy(), s[want])
    dt.dt_threshold_noalloc(snr[:0], hits[:0], 1.0, 2, idx[:0], val[:0], nf)
    torch.cuda.synchronize()
    assert int(nf.item()) == 0
