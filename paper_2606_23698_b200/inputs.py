"""Seeded synthetic input generators shared by the tests, the oracle legs and bench.py.

Holds none of the method's arithmetic: it only produces the complex128 arrays the
configs in BASELINE.json name. Counter-based, so any sub-block can be
regenerated: u(i) = (splitmix64(seed * 2^40 + i) >> 11) * 2^-53 with real index
i = 2 * flat + part.
"""
import numpy as np

_MASK = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x):
    x = (x + np.uint64(0x9E3779B97F4A7C15)) & _MASK
    z = x
    z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _MASK
    z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _MASK
    return z ^ (z >> np.uint64(31))


def uniform01(seed, start, count, stream=0):
    """count doubles in [0,1) for counters start .. start+count-1 of (seed, stream)."""
    with np.errstate(over="ignore"):
        i = np.arange(start, start + count, dtype=np.uint64)
        base = np.uint64((seed << 40) & 0xFFFFFFFFFFFFFFFF) + np.uint64((stream << 60) & 0xFFFFFFFFFFFFFFFF)
        z = _splitmix64(base + i)
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def _chunks(total, chunk=1 << 24):
    s = 0
    while s < total:
        c = min(chunk, total - s)
        yield s, c
        s += c


def uniform_pm1(shape, seed, out=None):
    """re, im iid uniform in [-1, 1) (configs 1, 4, 5)."""
    n = int(np.prod(shape))
    y = np.empty(2 * n, dtype=np.float64) if out is None else out.view(np.float64).reshape(-1)
    for s, c in _chunks(2 * n):
        y[s:s + c] = 2.0 * uniform01(seed, s, c) - 1.0
    return y.view(np.complex128).reshape(shape)


def loguniform(shape, seed, lo=-30, hi=30):
    """|re|, |im| = 2^(lo + (hi-lo) u), independent random signs (config 2)."""
    n = int(np.prod(shape))
    y = np.empty(2 * n, dtype=np.float64)
    for s, c in _chunks(2 * n):
        mag = np.exp2(lo + (hi - lo) * uniform01(seed, s, c, stream=0))
        sg = np.where(uniform01(seed, s, c, stream=1) < 0.5, -1.0, 1.0)
        y[s:s + c] = sg * mag
    return y.view(np.complex128).reshape(shape)


def normal(shape, seed):
    """re, im iid standard normal by Box-Muller from two uniform streams (config 3)."""
    n = int(np.prod(shape))
    y = np.empty(2 * n, dtype=np.float64)
    for s, c in _chunks(2 * n):
        u1 = 1.0 - uniform01(seed, s, c, stream=0)  # (0, 1]
        u2 = uniform01(seed, s, c, stream=1)
        y[s:s + c] = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return y.view(np.complex128).reshape(shape)


CONFIGS = {
    # name: (kind, shape, distribution, seed) -- BASELINE.json configs[0..4]
    "c1_32cubed": ("3d", (32, 32, 32), "uniform", 0),
    "c2_128cubed_lograng": ("3d", (128, 128, 128), "loguniform", 1),
    "c3_1d_1024x65536": ("1d", (65536, 1024), "normal", 2),
    "c4_512cubed": ("3d", (512, 512, 512), "uniform", 3),
    "c5_1024cubed": ("3d", (1024, 1024, 1024), "uniform", 4),
}


def make(dist, shape, seed):
    if dist == "uniform":
        return uniform_pm1(shape, seed)
    if dist == "loguniform":
        return loguniform(shape, seed)
    if dist == "normal":
        return normal(shape, seed)
    raise ValueError(dist)
