"""Counter-based seeded random numbers for the synthetic workloads.

This module holds NO arithmetic of the paper's method.  It only turns
(seed, linear index) into reproducible numbers, so that the fp64 CPU oracle
(`oracle/`) and the CUDA path (`paper_2401_06755_b200/`) can be fed the very
same inputs without sharing any code of the method itself.

Generator: SplitMix64 evaluated at counter `seed * 2^40 + index` (one state
per array element, no sequential state), so values do not depend on numpy's
version, on chunking, or on thread counts.
"""
from __future__ import annotations

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def splitmix64(counter: np.ndarray) -> np.ndarray:
    """SplitMix64 output function applied element-wise to uint64 counters."""
    with np.errstate(over="ignore"):
        z = (counter + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        z = z ^ (z >> np.uint64(31))
    return z


def _counters(seed: int, n: int, stream: int = 0) -> np.ndarray:
    base = (np.uint64(seed) << np.uint64(40)) ^ (np.uint64(stream) << np.uint64(36))
    with np.errstate(over="ignore"):
        return base + np.arange(n, dtype=np.uint64)


def uniform01(seed: int, n: int, stream: int = 0) -> np.ndarray:
    """n doubles in the open interval (0, 1): (top 53 bits + 0.5) / 2^53."""
    bits = splitmix64(_counters(seed, n, stream)) >> np.uint64(11)
    return (bits.astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def uniform(seed: int, n: int, lo: float = -1.0, hi: float = 1.0) -> np.ndarray:
    return lo + (hi - lo) * uniform01(seed, n)


def normal(seed: int, n: int) -> np.ndarray:
    """n standard normals by Box-Muller from two independent counter streams."""
    u1 = uniform01(seed, n, stream=1)
    u2 = uniform01(seed, n, stream=2)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
