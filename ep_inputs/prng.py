"""Counter-based seeded PRNG (splitmix64) for the synthetic input generators.

This module holds no arithmetic of the method ("All generators use an in-repo
PRNG"); it only turns (seed, counter) into reproducible uniform numbers so that meshes are
bit-reproducible on any machine and with any numpy version.
"""
from __future__ import annotations

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def splitmix64(seed: int, counter: np.ndarray) -> np.ndarray:
    """splitmix64 output function applied to (seed + (counter+1) * golden-gamma), vectorised."""
    with np.errstate(over="ignore"):
        c = np.asarray(counter, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + (c + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, counter: np.ndarray) -> np.ndarray:
    """Uniform doubles in [0,1) with 53 random bits."""
    z = splitmix64(seed, counter)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def uniform(seed: int, counter: np.ndarray, lo: float, hi: float) -> np.ndarray:
    return lo + (hi - lo) * uniform01(seed, counter)
