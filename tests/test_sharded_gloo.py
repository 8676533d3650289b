"""Exposure-sharded search: the host logic -- slices, the
variable-length all-gather of the sparse per-orbit partial sums, the rank-ordered merge -- on CPU with gloo,
world_size 2 and 3.  The partial sums come from the oracle evaluated on each rank's exposure slice; the merged result
must equal the oracle on the whole survey (hits exactly, SNR to the rounding of a re-associated fp64 sum) and be
bit-identical on every rank."""
import multiprocessing as mp
import socket

import numpy as np
import pytest

import dtsynth as ds
import oracle
from paper_2503_08854_b200.sharded import exposure_slices


def merge_lists(n, lists):
    """What dt_partials_reset + dt_partials_add do on the device, written out: sums over the lists in order."""
    S, Wt, hits = np.zeros(n), np.zeros(n), np.zeros(n, np.int32)
    for idx, s, w, h in lists:
        idx = np.asarray(idx, dtype=np.int64)
        S[idx] += np.asarray(s, dtype=np.float64)
        Wt[idx] += np.asarray(w, dtype=np.float64)
        hits[idx] += np.asarray(h, dtype=np.int32)
    return S, Wt, hits


def _scene():
    cfg = ds.focused(ds.scaled(ds.CONFIGS["small_mba"], n_orbits=1500, n_exp=41, width=96, height=80))
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    flux = [sc.flux_plane_np(j) for j in range(cfg.n_exp)]
    return sc, flux


def _slice_partials(sc, flux, lo, hi):
    sub = oracle.Survey(sc.t[lo:hi], sc.obs_ecl[lo:hi], sc.ra0[lo:hi], sc.dec0[lo:hi], sc.cfg.width, sc.cfg.height,
                        sc.pixel_scale, sc.gm, sc.c, sc.obliquity, 0, sc.var_scalar[lo:hi])
    r = oracle.stack(sub, flux[lo:hi], None, sc.elements(), sc.t0)
    idx = np.flatnonzero(r["hits"] > 0).astype(np.int64)
    return idx, r["S"][idx], r["Wt"][idx], r["hits"][idx].astype(np.int32)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import os
    import torch
    import torch.distributed as dist
    from paper_2503_08854_b200.sharded import exchange_partials
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        sc, flux = _scene()
        lo, hi = exposure_slices(sc.cfg.n_exp, world)[rank]
        local = tuple(torch.from_numpy(np.ascontiguousarray(x)) for x in _slice_partials(sc, flux, lo, hi))
        lists = exchange_partials(local)
        S, Wt, hits = merge_lists(sc.cfg.n_orbits, [tuple(t.numpy() for t in part) for part in lists])
        q.put((rank, [int(p[0].numel()) for p in lists], S, Wt, hits))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_sparse_partial_sum_exchange(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = {}
    for _ in range(world):
        r = q.get(timeout=300)
        out[r[0]] = r[1:]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    sc, flux = _scene()
    full = oracle.stack(oracle.Survey.from_scene(sc), flux, None, sc.elements(), sc.t0)
    sizes0, S0, Wt0, hits0 = out[0]
    assert sum(sizes0) > 0 and all(s < sc.cfg.n_orbits for s in sizes0), "the lists are sparse"
    for r in range(1, world):                       # every rank ends with the same bits
        assert out[r][0] == sizes0
        assert np.array_equal(out[r][1], S0) and np.array_equal(out[r][2], Wt0) and np.array_equal(out[r][3], hits0)
    assert np.array_equal(hits0, full["hits"])
    assert np.allclose(S0, full["S"], rtol=1e-12, atol=1e-13) and np.allclose(Wt0, full["Wt"], rtol=1e-12)
    snr = np.where(hits0 > 0, S0 / np.sqrt(np.where(Wt0 > 0, Wt0, 1.0)), 0.0)
    assert np.all(np.abs(snr - full["snr"]) <= 1e-9 * np.maximum(np.abs(full["snr"]), 1e-3))


def test_exposure_slices_partition_the_survey():
    for n, w in [(41, 2), (41, 3), (8, 8), (1000, 7)]:
        sl = exposure_slices(n, w)
        assert sl[0][0] == 0 and sl[-1][1] == n and all(a[1] == b[0] for a, b in zip(sl, sl[1:]))
        sizes = [hi - lo for lo, hi in sl]
        assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1
    with pytest.raises(ValueError):
        exposure_slices(3, 4)
