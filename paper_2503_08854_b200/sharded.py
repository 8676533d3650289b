"""Exposure-sharded search over the ranks of a torch.distributed group.

The paper's partitioning ("images are partitioned across nodes without replication"):
every rank holds a slice of the exposures, searches ALL candidate orbits against its slice, and because "the results
of these computations are extremely sparse" only the orbits with valid intersections travel.  Here

    rank r:  dt_stack over its exposure slice          (kernels 1-3; dtrack.h)
             dt_partials_sparse                        (device compaction: index, S, Wt, hits of the orbits with hits)
    all:     ONE variable-length all-gather of those lists                      (this file: plumbing only)
    rank r:  dt_partials_reset; dt_partials_add(list of rank 0), (rank 1), ...; dt_partials_finalize

so that every rank ends with the same per-orbit SNR (the lists are added in ascending rank = ascending exposure
order on every rank: same operations, same order, same bits) and dt_topk / dt_threshold work on any of them.  The
slices are contiguous and ascending, so the result is the plain stack up to the re-association of fp64 sums.
Nothing here computes: the arithmetic is in the library's kernels; `exchange_partials` moves tensors with the group's
backend (NCCL for CUDA tensors on NVLink; gloo for the CPU tests of the host logic).
"""
from __future__ import annotations

from typing import List, Tuple

import numpy as np


def exposure_slices(n_exposures: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous, ascending, balanced [lo, hi) per rank; every exposure in exactly one slice."""
    if world < 1 or n_exposures < world:
        raise ValueError("need at least one exposure per rank")
    base, extra = divmod(n_exposures, world)
    out, lo = [], 0
    for r in range(world):
        hi = lo + base + (1 if r < extra else 0)
        out.append((lo, hi))
        lo = hi
    return out


def exchange_partials(local, group=None):
    """local = (index int64 [m], S f64 [m], Wt f64 [m], hits i32 [m]) torch tensors of this rank (CPU for gloo, CUDA
    for NCCL).  -> the lists of all ranks, in rank order.  One all_gather of the lengths, one of each padded field."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    idx, S, Wt, hits = local
    dev = idx.device
    m = torch.tensor([idx.numel()], dtype=torch.int64, device=dev)
    sizes = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(sizes, m, group=group)
    sizes = [int(s.item()) for s in sizes]
    cap = max(max(sizes), 1)

    def gather(x):
        pad = torch.zeros(cap, dtype=x.dtype, device=dev)
        pad[:x.numel()] = x
        bufs = [torch.empty(cap, dtype=x.dtype, device=dev) for _ in range(world)]
        dist.all_gather(bufs, pad, group=group)
        return bufs

    gi, gs, gw, gh = gather(idx), gather(S), gather(Wt), gather(hits)
    return [(gi[r][:sizes[r]], gs[r][:sizes[r]], gw[r][:sizes[r]], gh[r][:sizes[r]]) for r in range(world)]


class ShardedTracker:
    """One rank of an exposure-sharded search.  `scene_like` carries the FULL survey's metadata (t, obs_ecl, ra0, dec0,
    var_scalar, cfg.width/height/variance_mode, constants); this rank's context is created on its slice only."""

    def __init__(self, scene_like, rank: int, world: int, device: int = 0, group=None, **kw):
        from . import Tracker
        self.rank, self.world, self.group, self.device = rank, world, group, device
        self.lo, self.hi = exposure_slices(int(np.asarray(scene_like.t).size), world)[rank]
        sl = slice(self.lo, self.hi)
        cfg = scene_like.cfg
        kw.setdefault("variance_mode", cfg.variance_mode)
        kw.setdefault("var_scalar", np.asarray(scene_like.var_scalar)[sl])
        self.trk = Tracker(np.asarray(scene_like.t)[sl], np.asarray(scene_like.obs_ecl)[sl],
                           np.asarray(scene_like.ra0)[sl], np.asarray(scene_like.dec0)[sl], cfg.width, cfg.height,
                           scene_like.pixel_scale, gm=scene_like.gm, c=scene_like.c, obliquity=scene_like.obliquity,
                           device=device, **kw)

    def load_image_batch(self, first_exposure: int, flux, var=None):
        """first_exposure is an index of the FULL survey; the planes must belong to this rank's slice."""
        if not (self.lo <= first_exposure and first_exposure + int(flux.shape[0]) <= self.hi):
            raise ValueError("exposures [%d, %d) are not in this rank's slice [%d, %d)" %
                             (first_exposure, first_exposure + int(flux.shape[0]), self.lo, self.hi))
        self.trk.load_image_batch(first_exposure - self.lo, flux, var)

    def stack(self, elements, t0=0.0):
        """elements: torch CUDA tensor [n, 6] (the same on every rank).  -> (snr, hits) CUDA tensors, equal on all ranks."""
        from . import dt_partials_add, dt_partials_finalize, dt_partials_reset, dt_partials_sparse
        self.trk.stack(elements, t0)
        n = int(elements.shape[0])
        local = dt_partials_sparse(self.trk.ctx, n, device=elements.device)
        lists = exchange_partials(local, self.group) if self.world > 1 else [local]
        dt_partials_reset(self.trk.ctx)
        for part in lists:                      # ascending rank = ascending exposure slice: the summation order
            dt_partials_add(self.trk.ctx, *part)
        return dt_partials_finalize(self.trk.ctx, n, device=elements.device)

    def topk(self, k, min_hits=0):
        return self.trk.topk(k, min_hits)

    def threshold(self, snr_min, min_hits=0, max_out=1 << 20):
        return self.trk.threshold(snr_min, min_hits, max_out)

    def close(self):
        self.trk.close()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
