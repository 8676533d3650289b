"""N > 1 is "replicas only": every rank holds the images and processes its own
block of seeded orbits; the only cross-rank logic is the block assignment and the max-over-ranks of
the timings.  Both are exercised here with world_size 2 on the gloo backend (CPU)."""
import os
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist          # noqa: E402
import torch.multiprocessing as mp        # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    import dtsynth as ds
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = ds.scaled(ds.CONFIGS["small_mba"], n_orbits=1000)
    el = bench.rank_elements(cfg, rank, world)
    ms = bench.max_over_ranks([10.0 + rank, 5.0 - rank], world)
    dist.barrier()
    q.put((rank, el, ms))
    dist.destroy_process_group()


def test_rank_blocks_and_max_over_ranks():
    import dtsynth as ds
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = {}
    for _ in range(world):
        r, el, ms = q.get(timeout=120)
        got[r] = (el, ms)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    cfg = ds.scaled(ds.CONFIGS["small_mba"], n_orbits=1000)
    both = ds.elements(cfg, 0, 2000)
    assert np.array_equal(got[0][0], both[:1000]) and np.array_equal(got[1][0], both[1000:])
    assert not np.array_equal(got[0][0], got[1][0])
    for r in range(world):
        assert got[r][1] == [11.0, 5.0]          # MAX over ranks, on every rank


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5], 1) == [1.5, 2.5]
