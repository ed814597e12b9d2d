"""Exact results for the 2D Ising model on the L x L torus (and brute force on small 3D boxes).  TEST INFRASTRUCTURE (pins).

PAPER.md L137: "a wealth of exact or extremely accurate results are available for it as
reference points".  Two independent references:

* brute force: enumeration of all 2^(L*L) states for L = 4 (65 536 states) -> g(E, M),
  from which every population average of Eq. 3 (L77-L86) and ln Z follow exactly at any beta;
* Kaufman's closed form of the finite-torus partition function (ref. [28] context, L361),
  evaluated in the log domain with mpmath; energy and specific heat from derivatives.
  It is checked against the L = 4 enumeration in tests/test_exact_refs.py before it is used
  for L = 16 ... 256.

Nothing here is used by, or shares code with, the oracle's PA implementation or the CUDA path.
"""
import math
from functools import lru_cache

import mpmath as mp
import numpy as np


# ---------------------------------------------------------------------------------------------
# brute force
# ---------------------------------------------------------------------------------------------

def enumerate_states_j(L, Jx, Jy):
    """As enumerate_states for H = -sum_<ab> J_ab s_a s_b with couplings Jx[y*L+x] on the bond (x,y)-(x+1,y) and
    Jy[y*L+x] on the bond (x,y)-(x,y+1), periodic (the generalisation of PAPER.md L313)."""
    N = L * L
    assert N <= 20
    states = np.arange(1 << N, dtype=np.int64)
    spins = ((states[:, None] >> np.arange(N)[None, :]) & 1).astype(np.int8) * 2 - 1
    grid = spins.reshape(-1, L, L).astype(np.int64)
    jx = np.asarray(Jx, dtype=np.int64).reshape(1, L, L); jy = np.asarray(Jy, dtype=np.int64).reshape(1, L, L)
    E = -(jx * grid * np.roll(grid, -1, axis=2)).sum(axis=(1, 2)) - (jy * grid * np.roll(grid, -1, axis=1)).sum(axis=(1, 2))
    M = grid.sum(axis=(1, 2))
    return E.astype(np.int64), M.astype(np.int64)


def exact_small_j(beta, L, Jx, Jy):
    """Exact canonical averages of the +-J sample by enumeration."""
    N = L * L
    E, M = enumerate_states_j(L, Jx, Jy)
    Emin = E.min()
    w = np.exp(-beta * (E - Emin).astype(np.float64))
    p = w / w.sum()
    e1 = (p * E).sum(); e2 = (p * E.astype(np.float64) ** 2).sum()
    m = M.astype(np.float64) / N
    lnZ = math.log(w.sum()) - beta * Emin
    return {"e": e1 / N, "C": beta * beta * (e2 - e1 * e1) / N, "absm": (p * np.abs(m)).sum(), "m2": (p * m ** 2).sum(),
            "lnZ": lnZ, "betaF_per_N": -lnZ / N, "S_per_N": beta * e1 / N + lnZ / N,
            "pE": {int(v): float(p[E == v].sum()) for v in np.unique(E)}}


@lru_cache(maxsize=None)
def enumerate_states(L=4):
    """All 2^(L*L) states: returns (E, M) int arrays indexed by the state's bit pattern
    (bit s = spin at site s = y*L+x; 1 = up).  H = -sum_<ab> s_a s_b, periodic (Eq. 10)."""
    N = L * L
    assert N <= 20
    states = np.arange(1 << N, dtype=np.int64)
    spins = ((states[:, None] >> np.arange(N)[None, :]) & 1).astype(np.int8) * 2 - 1   # [2^N][N]
    grid = spins.reshape(-1, L, L)
    E = -(grid * np.roll(grid, -1, axis=2)).sum(axis=(1, 2)) - (grid * np.roll(grid, -1, axis=1)).sum(axis=(1, 2))
    M = grid.sum(axis=(1, 2))
    return E.astype(np.int64), M.astype(np.int64)


@lru_cache(maxsize=None)
def density_of_states(L=4):
    """g(E) as a dict {E: count}."""
    E, _ = enumerate_states(L)
    vals, cnt = np.unique(E, return_counts=True)
    return {int(v): int(c) for v, c in zip(vals, cnt)}


def exact_small(beta, L=4):
    """Exact canonical averages on the L x L torus by enumeration (the quantities of Eq. 3-5)."""
    N = L * L
    E, M = enumerate_states(L)
    Emin = E.min()
    w = np.exp(-beta * (E - Emin).astype(np.float64))
    Z = w.sum()
    p = w / Z
    e1 = (p * E).sum()
    e2 = (p * E.astype(np.float64) ** 2).sum()
    m = M.astype(np.float64) / N
    lnZ = math.log(Z) - beta * Emin
    return {
        "e": e1 / N,
        "C": beta * beta * (e2 - e1 * e1) / N,
        "absm": (p * np.abs(m)).sum(),
        "m2": (p * m ** 2).sum(),
        "m4": (p * m ** 4).sum(),
        "lnZ": lnZ,
        "betaF_per_N": -lnZ / N,
        "S_per_N": beta * e1 / N + lnZ / N,
        "pE": {int(v): float(p[E == v].sum()) for v in np.unique(E)},
    }


@lru_cache(maxsize=None)
def enumerate_box(dims):
    """All 2^N states of the periodic simple-cubic box dims = (Lx, Ly, Lz), N = Lx Ly Lz <= 20 (O16; PAPER.md L313,
    L43): (E, M) indexed by the bit pattern, bit s = spin at site s = (z*Ly + y)*Lx + x.  H = -sum_s s_s (s_{x+1} + s_{y+1} +
    s_{z+1}) with periodic neighbours: numpy.roll along an axis of length 2 returns the one other site for both directions, so
    that bond is counted once from each of its two sites (the "double bond" of a period-2 direction)."""
    Lx, Ly, Lz = dims
    N = Lx * Ly * Lz
    assert N <= 20
    states = np.arange(1 << N, dtype=np.int64)
    spins = ((states[:, None] >> np.arange(N)[None, :]) & 1).astype(np.int8) * 2 - 1
    g = spins.reshape(-1, Lz, Ly, Lx).astype(np.int64)
    E = -(g * (np.roll(g, -1, axis=3) + np.roll(g, -1, axis=2) + np.roll(g, -1, axis=1))).sum(axis=(1, 2, 3))
    M = g.sum(axis=(1, 2, 3))
    return E.astype(np.int64), M.astype(np.int64)


@lru_cache(maxsize=None)
def density_of_states_box(dims):
    E, _ = enumerate_box(dims)
    vals, cnt = np.unique(E, return_counts=True)
    return {int(v): int(c) for v, c in zip(vals, cnt)}


def exact_box(beta, dims):
    """Exact canonical averages (Eq. 3-5) on the periodic box by enumeration."""
    N = dims[0] * dims[1] * dims[2]
    E, M = enumerate_box(tuple(dims))
    Emin = E.min()
    w = np.exp(-beta * (E - Emin).astype(np.float64))
    Z = w.sum()
    p = w / Z
    e1 = (p * E).sum(); e2 = (p * E.astype(np.float64) ** 2).sum()
    m = M.astype(np.float64) / N
    lnZ = math.log(Z) - beta * Emin
    return {"e": e1 / N, "C": beta * beta * (e2 - e1 * e1) / N, "absm": (p * np.abs(m)).sum(), "m2": (p * m ** 2).sum(),
            "m4": (p * m ** 4).sum(), "lnZ": lnZ, "betaF_per_N": -lnZ / N, "S_per_N": beta * e1 / N + lnZ / N,
            "pE": {int(v): float(p[E == v].sum()) for v in np.unique(E)}}


# ---------------------------------------------------------------------------------------------
# Kaufman's finite-lattice partition function (B. Kaufman 1949; McCoy & Wu, ref. [28])
#   Z = 1/2 (2 sinh 2K)^(N/2) (Z1 + Z2 + Z3 + Z4),  K = beta J,
#   Z1 = prod_{r=0}^{L-1} 2 cosh(L g_{2r+1}/2),  Z2 = prod 2 sinh(L g_{2r+1}/2),
#   Z3 = prod_{r=0}^{L-1} 2 cosh(L g_{2r}/2),    Z4 = prod 2 sinh(L g_{2r}/2),
#   cosh g_l = cosh 2K coth 2K - cos(l pi / L)  (g_l > 0) for l >= 1,   g_0 = 2K + ln tanh K
#   (g_0 < 0 for K < K_c: keep the sign, it makes Z4 negative above T_c).
# ---------------------------------------------------------------------------------------------

def kaufman_lnZ(beta, L, dps=60):
    """ln Z of the L x L periodic Ising model (J = 1) at inverse temperature beta > 0 (mpmath mpf)."""
    with mp.workdps(dps):
        K = mp.mpf(beta)
        N = L * L
        if K == 0:
            return N * mp.log(2)
        c2, s2 = mp.cosh(2 * K), mp.sinh(2 * K)

        def gamma(l):
            if l == 0:
                return 2 * K + mp.log(mp.tanh(K))
            return mp.acosh(c2 * c2 / s2 - mp.cos(mp.pi * l / L))

        Z1 = Z2 = Z3 = Z4 = mp.mpf(1)
        for r in range(L):
            go, ge = gamma(2 * r + 1), gamma(2 * r)
            Z1 *= 2 * mp.cosh(L * go / 2)
            Z2 *= 2 * mp.sinh(L * go / 2)
            Z3 *= 2 * mp.cosh(L * ge / 2)
            Z4 *= 2 * mp.sinh(L * ge / 2)
        return mp.log(mp.mpf(1) / 2) + (mp.mpf(N) / 2) * mp.log(2 * s2) + mp.log(Z1 + Z2 + Z3 + Z4)


def kaufman(beta, L, dps=60, h=None):
    """Exact ln Z, energy per site e = -(1/N) d lnZ / d beta and specific heat per site
    C = (beta^2/N) d^2 lnZ / d beta^2 (central differences at high precision)."""
    N = L * L
    with mp.workdps(dps):
        b = mp.mpf(beta)
        h = mp.mpf(10) ** (-12) if h is None else mp.mpf(h)
        f0, fp, fm = kaufman_lnZ(b, L, dps), kaufman_lnZ(b + h, L, dps), kaufman_lnZ(b - h, L, dps)
        d1 = (fp - fm) / (2 * h)
        d2 = (fp - 2 * f0 + fm) / (h * h)
        return {"lnZ": float(f0), "e": float(-d1 / N), "C": float(b * b * d2 / N),
                "betaF_per_N": float(-f0 / N), "S_per_N": float((-b * d1 + f0) / N)}


BETA_C = 0.5 * math.log(1.0 + math.sqrt(2.0))   # L137
