"""Counter-based, platform-independent random numbers for the synthetic workloads.

Every draw is a pure function of (seed, stream, index), so any sub-range of any array can be
regenerated anywhere (CPU numpy, torch on CPU, torch on CUDA) and gives the same bits
("Randomness").  The integer part is exact by construction; the two
floating-point recipes below are made reproducible as follows:

* uniforms  u = ((h >> 11) + 0.5) * 2**-53   in (0, 1): exact in fp64 (one int->double conversion,
  one add of 0.5 that is exact below 2**53, one power-of-two scaling).
* normals   Box-Muller in fp64, then QUANTISED to a grid of 2**-16:  z = rint(g * 65536) / 65536.
  numpy's and torch's log/cos may differ in the last fp64 ulp; after quantisation the two agree
  unless g*65536 lies within ~1e-11 of a half-integer (probability ~1e-11 per draw).  Quantised
  values have at most 3+16 significant bits, so they are exact in fp32.

This module contains NO arithmetic of the tracking method (no Kepler, no projection).

Constants (fixed once, written here so that both backends and any reader agree):
  GOLDEN = 0x9E3779B97F4A7C15,  M1 = 0xBF58476D1CE4E5B9,  M2 = 0x94D049BB133111EB
  mix64(x): x ^= x >> 30; x *= M1; x ^= x >> 27; x *= M2; x ^= x >> 31      (all mod 2**64)
  key(seed, stream)  = mix64(mix64(seed * GOLDEN + 1) + stream * GOLDEN)
  h(seed, stream, k) = mix64(key(seed, stream) + (k + 1) * GOLDEN)
"""
from __future__ import annotations

import numpy as np

GOLDEN = 0x9E3779B97F4A7C15
M1 = 0xBF58476D1CE4E5B9
M2 = 0x94D049BB133111EB
_MASK = (1 << 64) - 1
NORMAL_QUANTUM = 65536.0  # normals live on a grid of 1/65536

# Stream identifiers (one independent stream per generated quantity).
STREAM_A, STREAM_E, STREAM_I, STREAM_NODE, STREAM_PERI, STREAM_M0 = 1, 2, 3, 4, 5, 6
STREAM_TIME, STREAM_TAN_LON, STREAM_TAN_LAT, STREAM_DITHER_X, STREAM_DITHER_Y = 10, 11, 12, 13, 14
STREAM_VAR, STREAM_AMP, STREAM_PLACE = 20, 21, 22
STREAM_NOISE_BASE = 1 << 20  # + exposure index (first Box-Muller uniform)
STREAM_NOISE_BASE2 = 1 << 21  # + exposure index (second Box-Muller uniform)


def _mix64_int(x: int) -> int:
    x &= _MASK
    x ^= x >> 30
    x = (x * M1) & _MASK
    x ^= x >> 27
    x = (x * M2) & _MASK
    x ^= x >> 31
    return x


def stream_key(seed: int, stream: int) -> int:
    """Python-int key of a (seed, stream) pair; shared by the numpy and torch paths."""
    return _mix64_int(_mix64_int(seed * GOLDEN + 1) + stream * GOLDEN)


# ----------------------------------------------------------------------------------------------
# numpy backend
# ----------------------------------------------------------------------------------------------
def _mix64_np(x: np.ndarray) -> np.ndarray:
    x = x.copy()
    x ^= x >> np.uint64(30)
    x *= np.uint64(M1)
    x ^= x >> np.uint64(27)
    x *= np.uint64(M2)
    x ^= x >> np.uint64(31)
    return x


def hash_np(seed: int, stream: int, k) -> np.ndarray:
    """h(seed, stream, k) for an array (or scalar) of indices k >= 0 -> uint64."""
    k = np.asarray(k, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = np.uint64(stream_key(seed, stream)) + (k + np.uint64(1)) * np.uint64(GOLDEN)
        return _mix64_np(np.atleast_1d(x)).reshape(k.shape)


def uniform_np(seed: int, stream: int, k) -> np.ndarray:
    """u in (0, 1), fp64, exact on every platform."""
    h = hash_np(seed, stream, k)
    return ((h >> np.uint64(11)).astype(np.float64) + 0.5) * (2.0 ** -53)


def normal_np(seed: int, stream1: int, stream2: int, k) -> np.ndarray:
    """Quantised standard normal (grid 2**-16), fp64 holding fp32-exact values."""
    u1 = uniform_np(seed, stream1, k)
    u2 = uniform_np(seed, stream2, k)
    g = np.sqrt(-2.0 * np.log(u1)) * np.cos((2.0 * np.pi) * u2)
    return np.rint(g * NORMAL_QUANTUM) / NORMAL_QUANTUM


# ----------------------------------------------------------------------------------------------
# torch backend (CPU or CUDA): same bits, int64 two's-complement arithmetic
# ----------------------------------------------------------------------------------------------
def _s64(v: int) -> int:
    v &= _MASK
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr_t(x, s: int):
    # logical shift right of an int64 tensor
    return (x >> s) & ((1 << (64 - s)) - 1)


def _mix64_t(x):
    x = x ^ _lsr_t(x, 30)
    x = x * _s64(M1)
    x = x ^ _lsr_t(x, 27)
    x = x * _s64(M2)
    x = x ^ _lsr_t(x, 31)
    return x


def hash_t(seed: int, stream: int, k):
    """torch version of hash_np; k is an int64 tensor of indices >= 0. Returns int64 (bit pattern)."""
    x = (k + 1) * _s64(GOLDEN) + _s64(stream_key(seed, stream))
    return _mix64_t(x)


def uniform_t(seed: int, stream: int, k):
    import torch

    h = hash_t(seed, stream, k)
    return (_lsr_t(h, 11).to(torch.float64) + 0.5) * (2.0 ** -53)


def normal_t(seed: int, stream1: int, stream2: int, k):
    import math

    import torch

    u1 = uniform_t(seed, stream1, k)
    u2 = uniform_t(seed, stream2, k)
    g = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)
    return torch.round(g * NORMAL_QUANTUM) / NORMAL_QUANTUM
