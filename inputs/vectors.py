"""Counter-based start-vector generator v0[J] = g(seed, J) in uniform[-1, 1).

PAPER.md:119 asks for "a random initial vector of norm 1"; BASELINE.json fixes
it to a seeded uniform[-1,1) vector, normalised.  A counter-based generator
lets any single element be produced without materialising the vector, which
the sampled-row parity check on the 2.4e9-element config needs
(reading Q13).

g(seed, J): z = seed + (J+1)*0x9E3779B97F4A7C15 (mod 2^64), followed by the
public-domain splitmix64 finaliser; the top 53 bits give u in [0,1) and the
value is 2u-1, an exactly representable double.  The same bits are produced by
the numpy (uint64) and the torch (int64, wrapping) implementation; a CPU test
checks that.
"""
from __future__ import annotations

import numpy as np

_GOLD = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB
_MASK64 = (1 << 64) - 1


def _g_scalar(seed: int, j: int) -> float:
    z = (seed + (j + 1) * _GOLD) & _MASK64
    z = ((z ^ (z >> 30)) * _M1) & _MASK64
    z = ((z ^ (z >> 27)) * _M2) & _MASK64
    z = z ^ (z >> 31)
    return (z >> 11) * (2.0 ** -52) - 1.0


def g_uniform(seed: int, idx) -> np.ndarray:
    """g(seed, idx) for an integer array (or scalar) of element indices, fp64."""
    j = np.asarray(idx, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & _MASK64) + (j + np.uint64(1)) * np.uint64(_GOLD)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(_M1)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(_M2)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -52) - 1.0


def start_vector_np(seed: int, dim: int, chunk: int = 1 << 24) -> np.ndarray:
    """Un-normalised v0 (fp64, length dim) on the host."""
    out = np.empty(dim, dtype=np.float64)
    for lo in range(0, dim, chunk):
        hi = min(dim, lo + chunk)
        out[lo:hi] = g_uniform(seed, np.arange(lo, hi, dtype=np.uint64))
    return out


def _s64(x: int) -> int:
    """Two's-complement reinterpretation of a 64-bit pattern as a signed int."""
    x &= _MASK64
    return x - (1 << 64) if x >= (1 << 63) else x


def start_vector_torch(seed: int, dim: int, device, dtype=None, chunk: int = 1 << 26):
    """Un-normalised v0 on a torch device, same bits as `start_vector_np`.

    Uses int64 arithmetic (wrapping multiply, masked shifts for the logical
    right shifts).  Generated in fp64 per chunk, then cast to `dtype`
    (default fp64).  Only plumbing: this is input generation, not the method.
    """
    import torch

    dtype = dtype or torch.float64
    out = torch.empty(dim, dtype=dtype, device=device)

    def lsr(z, k):
        return (z >> k) & ((1 << (64 - k)) - 1)

    for lo in range(0, dim, chunk):
        hi = min(dim, lo + chunk)
        j = torch.arange(lo + 1, hi + 1, dtype=torch.int64, device=device)
        z = j * _s64(_GOLD) + _s64(seed)
        z = (z ^ lsr(z, 30)) * _s64(_M1)
        z = (z ^ lsr(z, 27)) * _s64(_M2)
        z = z ^ lsr(z, 31)
        u = lsr(z, 11).to(torch.float64) * (2.0 ** -52) - 1.0
        out[lo:hi] = u.to(dtype)
    return out


def sample_indices(seed: int, dim: int, n: int) -> np.ndarray:
    """n seeded element indices in [0, dim), always including 0 and dim-1,
    sorted and unique (so the count can be slightly below n)."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    idx = rng.integers(0, dim, size=max(0, n - 2), dtype=np.int64)
    idx = np.concatenate([idx, np.array([0, dim - 1], dtype=np.int64)])
    return np.unique(idx)
