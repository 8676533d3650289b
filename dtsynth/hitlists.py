"""Controlled hit lists for the kernel-3 (gather + stack) micro-benchmarks.

Builds, on a CUDA device with torch, a hit list in the library's hit-list format (see
include/dtrack.h, dt_gather_hits) in which every (orbit, exposure) pair is a hit with probability
`density` and the hit pixel is drawn uniformly from a `cluster` x `cluster` window whose centre
moves from exposure to exposure:
    cluster = image size   -> regime L0 (uniform random pixels, one 32-B sector per 4-B payload)
    cluster = a few 100 px -> regime L1 (hits clustered as in a focused search)
    cluster = tens of px   -> regime L2 (many orbits per pixel: reuse)
No arithmetic of the tracking method lives here (pure index bookkeeping and random draws).
"""
from __future__ import annotations

from . import rng


def build(n_orbits: int, n_groups: int, width: int, height: int, cluster: int, density: float,
          seed: int, device, px_per_sector: int = 8):
    """-> dict(mask [G, n_pad] int32, base [G, n_pad/32] int64, offsets [hits] int32, hits,
    unique_sectors, touched_orbits) -- all torch tensors on `device`."""
    import torch

    n_pad = (n_orbits + 31) // 32 * 32
    tiles = n_pad // 32
    G = n_groups
    plane = width * height
    gen = torch.Generator(device=device)
    gen.manual_seed(int(rng.stream_key(seed, 99) & 0x7FFFFFFF))
    bits = torch.zeros((G, n_pad), dtype=torch.int64, device=device)
    for b in range(32):
        if density >= 1.0:
            on = torch.ones((G, n_pad), dtype=torch.bool, device=device)
        else:
            on = torch.rand((G, n_pad), device=device, generator=gen) < density
        on[:, n_orbits:] = False
        bits |= on.to(torch.int64) << b
    # hits of warp-tile w (32 consecutive orbits) in exposure (g, b): [G, tiles, 32]
    cnt_gtb = torch.stack([((bits >> b) & 1).reshape(G, tiles, 32).sum(2) for b in range(32)], dim=2)
    tile_tot = cnt_gtb.sum(2)                                            # [G, tiles]
    base = (torch.cumsum(tile_tot.reshape(-1), 0) - tile_tot.reshape(-1)).reshape(G, tiles).contiguous()
    seg = base.unsqueeze(2) + torch.cumsum(cnt_gtb, 2) - cnt_gtb         # start of exposure b's run
    hits = int(tile_tot.sum().item())
    # per hit: a random pixel of the window; block order = exposure-ascending, then lane-ascending
    offsets = torch.empty(max(hits, 1), dtype=torch.int32, device=device)
    sectors = 0
    cl = min(cluster, width, height)
    for g in range(G):
        bg = bits[g]
        sec_ids = []
        for b in range(32):
            on2 = ((bg >> b) & 1).reshape(tiles, 32)
            on = on2.bool().reshape(-1)
            k = int(on.sum().item())
            if k == 0:
                continue
            j = 32 * g + b
            cx = int((rng.stream_key(seed, 1000 + j) >> 8) % (width - cl + 1))
            cy = int((rng.stream_key(seed, 5000 + j) >> 8) % (height - cl + 1))
            px = cx + torch.randint(0, cl, (k,), device=device, generator=gen)
            py = cy + torch.randint(0, cl, (k,), device=device, generator=gen)
            off = py * width + px
            lane_rank = torch.cumsum(on2, 1) - on2
            pos = (seg[g, :, b].unsqueeze(1) + lane_rank).reshape(-1)[on]
            offsets[pos] = (off + (b << 27)).to(torch.int32)      # entry = (exposure in group) << 27 | pixel offset
            sec_ids.append(torch.unique((j * plane + off) // px_per_sector))   # 8 fp32 (4 float2) per 32-B sector
        if sec_ids:
            sectors += int(sum(s.numel() for s in sec_ids))               # exposures are disjoint
    cnt = tile_tot
    mask = (bits & 0xFFFFFFFF)
    mask = torch.where(mask >= (1 << 31), mask - (1 << 32), mask).to(torch.int32).contiguous()
    touched = int((bits != 0).any(0).sum().item())
    return dict(mask=mask, base=base, offsets=offsets, hits=hits, unique_sectors=sectors,
                touched_orbits=touched, n_pad=n_pad)
