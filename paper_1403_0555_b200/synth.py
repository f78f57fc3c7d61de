"""Seeded synthetic gauge orbits (link-angle fields) for the five BASELINE configs.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: it only draws link angles theta_{i,mu}.  It has its own (numpy) Philox4x32-10; the random
STARTS of the relaxation are generated inside each implementation (oracle and CUDA each carry their own
copy of the counter-based generator).

The paper's workloads are themselves synthetic: random ("hot", beta = 0) orbits whose seeds are not
published, so these stand in for them with the same distribution; the
Gaussian-plus-random-gauge-transform orbits of configs 2 and 4 come from BASELINE.json.  Recipe
(DESIGN.md section 5):

  key (seed, V); 53-bit uniform u from words (x0 | x1<<32) >> 11 of the Philox block
  tag 2  uniform links    counter (i*d+mu, 0, 0, 2):  theta = -pi + 2 pi u
  tag 3  Gaussian links   counter (i*d+mu, 0, 0, 3):  z = sqrt(-2 ln(1-u1)) cos(2 pi u2), u1 from words 0-1,
                                                       u2 from words 2-3;  theta = sigma z
  tag 4  gauge angles     counter (i, 0, 0, 4):        h_i = -pi + 2 pi u;
                                                       theta <- wrap(theta + h_i - h_{i+mu}) into [-pi, pi)
  site index i = x0 + N0*(x1 + N1*(x2 + N2*x3)); theta stored at [i*d + mu].
"""
from __future__ import annotations

import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = 0x9E3779B9
_W1 = 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Vectorised Philox4x32-10 (Salmon et al. 2011).  Counter words are uint64 arrays holding 32-bit
    values; returns four uint64 arrays of 32-bit words."""
    c0, c1, c2, c3 = (np.asarray(c, dtype=np.uint64) & _MASK for c in np.broadcast_arrays(c0, c1, c2, c3))
    k0 = int(k0) & 0xFFFFFFFF
    k1 = int(k1) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        hi0, lo0 = p0 >> _S32, p0 & _MASK
        hi1, lo1 = p1 >> _S32, p1 & _MASK
        c0, c1, c2, c3 = hi1 ^ c1 ^ np.uint64(k0), lo1, hi0 ^ c3 ^ np.uint64(k1), lo0
        k0 = (k0 + _W0) & 0xFFFFFFFF
        k1 = (k1 + _W1) & 0xFFFFFFFF
    return c0, c1, c2, c3


def _u53(lo, hi):
    r = ((hi << _S32) | lo) >> np.uint64(11)
    return r.astype(np.float64) * 2.0 ** -53


def volume(extents) -> int:
    return int(np.prod(np.asarray(extents, dtype=np.int64)))


def forward_neighbour(extents, mu):
    """Index of i + mu^ for every site (periodic)."""
    ext = [int(n) for n in extents]
    V = volume(ext)
    i = np.arange(V, dtype=np.int64)
    stride = int(np.prod(ext[:mu], dtype=np.int64)) if mu else 1
    x = (i // stride) % ext[mu]
    return i + (((x + 1) % ext[mu]) - x) * stride


def uniform_links(extents, seed):
    """Hot orbit: theta iid uniform[-pi, pi) (tag 2)."""
    d = len(extents)
    V = volume(extents)
    n = np.arange(V * d, dtype=np.uint64)
    w = philox4x32_10(n, 0, 0, 2, seed, V)
    return -np.pi + 2.0 * np.pi * _u53(w[0], w[1])


def gaussian_links(extents, seed, sigma):
    """theta = sigma * N(0,1) noise on the identity (tag 3, Box-Muller)."""
    d = len(extents)
    V = volume(extents)
    n = np.arange(V * d, dtype=np.uint64)
    w = philox4x32_10(n, 0, 0, 3, seed, V)
    u1 = _u53(w[0], w[1])
    u2 = _u53(w[2], w[3])
    return sigma * np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)


def gauge_angles(extents, seed):
    """h_i iid uniform[-pi, pi) (tag 4)."""
    V = volume(extents)
    w = philox4x32_10(np.arange(V, dtype=np.uint64), 0, 0, 4, seed, V)
    return -np.pi + 2.0 * np.pi * _u53(w[0], w[1])


def wrap(theta):
    """Wrap angles into [-pi, pi)."""
    t = np.mod(theta + np.pi, 2.0 * np.pi) - np.pi
    t[t >= np.pi] = -np.pi
    return t


def gauge_transform_links(extents, theta, h):
    """theta_{i,mu} <- wrap(theta_{i,mu} + h_i - h_{i+mu})."""
    d = len(extents)
    t = np.array(theta, dtype=np.float64).reshape(-1, d).copy()
    for mu in range(d):
        t[:, mu] += h - h[forward_neighbour(extents, mu)]
    return wrap(t.reshape(-1))


def gaussian_gauged_links(extents, seed, sigma):
    """Configs 2 and 4: Gaussian(sigma) noise on the identity, then a random gauge transformation."""
    return gauge_transform_links(extents, gaussian_links(extents, seed, sigma), gauge_angles(extents, seed))


def cold_links(extents):
    """Trivial (cold) orbit: all link angles zero."""
    return np.zeros(volume(extents) * len(extents))


# The five BASELINE.json configs.  `orbits` is a list of (extents, theta-factory, start seed, n_starts).
CONFIGS = {
    1: dict(name="cfg1_2d_4x4_hot", omega=1.7, eps=1e-13, max_sweeps=20000,
            orbits=[dict(extents=(4, 4), kind="uniform", seed=1, n_starts=4096)]),
    2: dict(name="cfg2_2d_8x8_gauss0.6", omega=1.7, eps=1e-13, max_sweeps=20000,
            orbits=[dict(extents=(8, 8), kind="gauss", sigma=0.6, seed=2, n_starts=1 << 20)]),
    3: dict(name="cfg3_3d_4x4x4_hot_x8", omega=1.7, eps=1e-13, max_sweeps=20000,
            orbits=[dict(extents=(4, 4, 4), kind="uniform", seed=s, n_starts=1 << 20) for s in range(3, 11)]),
    4: dict(name="cfg4_4d_4x4x4x4_gauss0.8", omega=1.7, eps=1e-13, max_sweeps=20000,
            orbits=[dict(extents=(4, 4, 4, 4), kind="gauss", sigma=0.8, seed=11, n_starts=1 << 22)]),
    5: dict(name="cfg5_4d_scan_hot", omega=1.7, eps=1e-12, max_sweeps=20000,
            orbits=[dict(extents=(n,) * 4, kind="uniform", seed=12, n_starts=(1 << 16) if n == 8 else (1 << 20))
                    for n in (2, 3, 4, 6, 8)]),
}


def make_theta(orbit: dict):
    ext = orbit["extents"]
    if orbit["kind"] == "uniform":
        return uniform_links(ext, orbit["seed"])
    if orbit["kind"] == "gauss":
        return gaussian_gauged_links(ext, orbit["seed"], orbit["sigma"])
    if orbit["kind"] == "cold":
        return cold_links(ext)
    raise ValueError(orbit["kind"])
