"""Exact results for the 2D periodic square-lattice Ising model (J = k_B = 1) used to pin the oracle.

Nothing here comes from oracle/ or from the CUDA path: brute-force enumeration (numpy), Kaufman's
finite-lattice partition function and Onsager/Yang's infinite-lattice results (mpmath, 50 digits),
and a binned Monte-Carlo error estimate.  SURVEY.md section 8(c) pins 3-5 give the formulas.
"""
from __future__ import annotations

import numpy as np
import mpmath as mp

mp.mp.dps = 50


# --------------------------------------------------------------------------------------
# brute force: all 2^(L*L) states of a tiny periodic lattice (each site's East and South edge)
# --------------------------------------------------------------------------------------
def enumerate_states(L: int):
    """Return (E, M) int arrays over all 2^(L*L) states; E = -sum_i s_i (s_E(i) + s_S(i))."""
    n = L * L
    assert n <= 20
    states = np.arange(1 << n, dtype=np.int64)
    s = np.empty((n, 1 << n), dtype=np.int8)
    for i in range(n):
        s[i] = np.where((states >> i) & 1, 1, -1)
    E = np.zeros(1 << n, dtype=np.int64)
    for i in range(n):
        y, x = divmod(i, L)
        e = y * L + (x + 1) % L
        so = ((y + 1) % L) * L + x
        E -= s[i].astype(np.int64) * (s[e].astype(np.int64) + s[so].astype(np.int64))
    M = s.astype(np.int64).sum(axis=0)
    return E, M


def exact_small(L: int, T: float):
    """Exact <E>/N, <|m|>, <m^2>, C/N and Z for a tiny lattice, in 50-digit arithmetic."""
    E, M = enumerate_states(L)
    n = L * L
    levels, inv = np.unique(E, return_inverse=True)
    g = np.bincount(inv)
    absM = np.bincount(inv, weights=np.abs(M).astype(np.float64))       # exact: integers < 2^53
    M2 = np.bincount(inv, weights=(M.astype(np.float64) ** 2))
    beta = mp.mpf(1) / mp.mpf(T)
    w = [mp.e ** (-beta * int(e)) for e in levels]
    Z = sum(int(gi) * wi for gi, wi in zip(g, w))
    Em = sum(int(e) * int(gi) * wi for e, gi, wi in zip(levels, g, w)) / Z
    E2 = sum(int(e) ** 2 * int(gi) * wi for e, gi, wi in zip(levels, g, w)) / Z
    am = sum(mp.mpf(a) * wi for a, wi in zip(absM, w)) / Z / n
    m2 = sum(mp.mpf(a) * wi for a, wi in zip(M2, w)) / Z / (n * n)
    return {
        "u": Em / n, "abs_m": am, "m2": m2,
        "c": (E2 - Em ** 2) / (n * mp.mpf(T) ** 2), "Z": Z,
        "levels": {int(e): int(gi) for e, gi in zip(levels, g)},
    }


# --------------------------------------------------------------------------------------
# Kaufman (1949): exact partition function of the periodic L x L lattice
# --------------------------------------------------------------------------------------
def kaufman_lnZ(L: int, K):
    K = mp.mpf(K)
    def gamma(l):
        if l == 0:
            return 2 * K + mp.log(mp.tanh(K))          # negative above T_c: carries the sign
        return mp.acosh(mp.cosh(2 * K) * mp.coth(2 * K) - mp.cos(l * mp.pi / L))
    g = [gamma(l) for l in range(2 * L)]
    # four products, each kept as (sign, log|.|)
    def logprod(terms):
        sign, acc = 1, mp.mpf(0)
        for t in terms:
            if t < 0:
                sign = -sign
            acc += mp.log(abs(t))
        return sign, acc
    parts = [
        logprod([2 * mp.cosh(L * g[2 * r + 1] / 2) for r in range(L)]),
        logprod([2 * mp.sinh(L * g[2 * r + 1] / 2) for r in range(L)]),
        logprod([2 * mp.cosh(L * g[2 * r] / 2) for r in range(L)]),
        logprod([2 * mp.sinh(L * g[2 * r] / 2) for r in range(L)]),
    ]
    top = max(p[1] for p in parts)
    tot = sum(p[0] * mp.e ** (p[1] - top) for p in parts)
    return -mp.log(2) + (mp.mpf(L * L) / 2) * mp.log(2 * mp.sinh(2 * K)) + top + mp.log(tot)


def kaufman_u(L: int, T: float):
    """u_L = -(1/L^2) d lnZ_L / dK at K = 1/T (numerical derivative in extended precision)."""
    old = mp.mp.dps
    mp.mp.dps = 60
    try:
        K = mp.mpf(1) / mp.mpf(T)
        d = mp.diff(lambda k: kaufman_lnZ(L, k), K, h=mp.mpf(10) ** (-15))
        return -d / (L * L)
    finally:
        mp.mp.dps = old


def kaufman_c(L: int, T: float):
    old = mp.mp.dps
    mp.mp.dps = 60
    try:
        K = mp.mpf(1) / mp.mpf(T)
        d2 = mp.diff(lambda k: kaufman_lnZ(L, k), K, 2, h=mp.mpf(10) ** (-12))
        return K * K * d2 / (L * L)
    finally:
        mp.mp.dps = old


# --------------------------------------------------------------------------------------
# Onsager (1944) energy and Yang (1952) spontaneous magnetisation, L -> infinity
# --------------------------------------------------------------------------------------
def onsager_u(T: float):
    K = mp.mpf(1) / mp.mpf(T)
    k = 2 * mp.sinh(2 * K) / mp.cosh(2 * K) ** 2
    return -mp.coth(2 * K) * (1 + (2 / mp.pi) * (2 * mp.tanh(2 * K) ** 2 - 1) * mp.ellipk(k * k))


def yang_m(T: float):
    K = mp.mpf(1) / mp.mpf(T)
    x = 1 - mp.sinh(2 * K) ** (-4)
    return x ** (mp.mpf(1) / 8) if x > 0 else mp.mpf(0)


# --------------------------------------------------------------------------------------
# Monte-Carlo error: binning
# --------------------------------------------------------------------------------------
def binned_mean_err(x, nbins: int = 50):
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nbins) * nbins
    b = x[:n].reshape(nbins, -1).mean(axis=1)
    return float(b.mean()), float(b.std(ddof=1) / np.sqrt(nbins))
