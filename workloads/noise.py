"""Counter-based Gaussian generator for the per-matvec noise model of
BASELINE.json configs[0] ("matvec error injected as Gaussian noise scaled to
relative 1e-4 ||AX||"; reading SURVEY.md S11).

The random numbers are an INPUT of the inexact operator, not part of the
method.  The CUDA library implements the same counter -> N(0,1) map (splitmix64
hash of (seed, apply index, row, column), Box-Muller) so both sides can draw the
same perturbation direction without exchanging arrays.
"""
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x):
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = x
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def counter_gaussian(seed, apply_index, m, n):
    """g[i, j] ~ N(0,1), a pure function of (seed, apply_index, i, j).

    key = splitmix64(splitmix64(seed ^ apply_index * 0xD1B54A32D192ED03) + i * n + j);
    u1 = (top 53 bits of key + 0.5) / 2^53, u2 from splitmix64(key);
    g = sqrt(-2 ln u1) cos(2 pi u2).
    """
    with np.errstate(over="ignore"):
        base = _splitmix64(np.uint64(seed) ^ ((np.uint64(apply_index) *
                                               np.uint64(0xD1B54A32D192ED03)) & _M64))
        idx = (np.arange(m, dtype=np.uint64)[:, None] * np.uint64(n)
               + np.arange(n, dtype=np.uint64)[None, :])
        k1 = _splitmix64((base + idx) & _M64)
        k2 = _splitmix64(k1)
    u1 = ((k1 >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)
    u2 = ((k2 >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
