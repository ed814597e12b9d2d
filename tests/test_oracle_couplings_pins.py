"""Pins of the oracle's bimodal-coupling workload (O15; "the case of different couplings including
spin glasses ... straightforward") against what the mathematics fixes (-m "not gpu")."""
import math

import numpy as np
import pytest

from oracle import exact_ising as ex
from oracle import pa_oracle as po
import pa_driver


def _random_j(L, seed):
    rng = np.random.default_rng(seed)
    return (rng.integers(0, 2, L * L) * 2 - 1).astype(np.int8), (rng.integers(0, 2, L * L) * 2 - 1).astype(np.int8)


def _mattis(L, seed):
    """Gauge couplings J_ab = eps_a eps_b: the ferromagnet in disguise."""
    rng = np.random.default_rng(seed)
    eps = (rng.integers(0, 2, (L, L)) * 2 - 1).astype(np.int8)
    Jx = eps * np.roll(eps, -1, axis=1); Jy = eps * np.roll(eps, -1, axis=0)
    return eps.reshape(-1), Jx.reshape(-1).astype(np.int8), Jy.reshape(-1).astype(np.int8)


@pytest.mark.parametrize("mode", [po.RNG_PHILOX, po.RNG_LCG])
def test_gauge_invariance_exact(mode):
    # sigma'_a = eps_a sigma_a, J'_ab = eps_a eps_b: every bond is satisfied in sigma' under J' iff it is in sigma under J = +1, the
    # acceptance depends on the number of unsatisfied bonds and on a random number keyed by (slot, site, sweep) only, so the Mattis
    # trajectory IS the gauge-transformed ferromagnetic trajectory, bit for bit; energies agree, magnetisations do not
    L, n = 6, 40
    eps, Jx, Jy = _mattis(L, 3)
    rng = np.random.default_rng(4)
    ferro = rng.integers(0, 2, (n, L * L), dtype=np.uint8)
    gauged = np.where(eps[None, :] > 0, ferro, 1 - ferro).astype(np.uint8)
    slots = np.arange(50, 50 + n)
    Ef, _ = po.energies_of(L, ferro)
    Eg, _ = po.energies_of_j(L, gauged, Jx, Jy)
    assert np.array_equal(Ef, Eg)
    po.sweep_slots(L, 9, 3, 0.4, 6, slots, ferro, rng_mode=mode)
    po.sweep_slots_j(L, 9, 3, 0.4, 6, slots, gauged, Jx, Jy, rng_mode=mode)
    assert np.array_equal(gauged, np.where(eps[None, :] > 0, ferro, 1 - ferro))
    assert np.array_equal(po.energies_of(L, ferro)[0], po.energies_of_j(L, gauged, Jx, Jy)[0])
    # all J = +1 through the coupling path = the plain ferromagnet
    a = rng.integers(0, 2, (n, L * L), dtype=np.uint8); b = a.copy()
    ones = np.ones(L * L, dtype=np.int8)
    po.sweep_slots(L, 9, 0, 0.3, 3, slots, a, rng_mode=mode); po.sweep_slots_j(L, 9, 0, 0.3, 3, slots, b, ones, ones, rng_mode=mode)
    assert np.array_equal(a, b)


def test_energies_with_couplings_bruteforce_and_level_offset():
    L = 4
    Jx, Jy = _random_j(L, 11)
    E, M = ex.enumerate_states_j(L, Jx, Jy)
    idx = np.random.default_rng(0).choice(1 << 16, 3000, replace=False)
    sp = ((idx[:, None] >> np.arange(16)[None, :]) & 1).astype(np.uint8)
    Eo, Mo = po.energies_of_j(L, sp, Jx, Jy)
    assert np.array_equal(Eo, E[idx]) and np.array_equal(Mo, M[idx])
    # every energy of the sample sits on one lattice of spacing 4: E = -2N + 4m + e0, e0 = 2 (number of J = -1 bonds) mod 4
    o = po.Oracle(L, 8, 1); o.set_couplings(Jx, Jy)
    e0 = o.level_offset
    assert e0 == (2 * int((Jx < 0).sum() + (Jy < 0).sum())) % 4
    assert np.all((E + 2 * 16 - e0) % 4 == 0)
    # an odd number of negative bonds: the other lattice
    Jx2 = Jx.copy(); Jx2[5] = -Jx2[5]
    o2 = po.Oracle(L, 8, 1); o2.set_couplings(Jx2, Jy)
    assert o2.level_offset == 2 - e0
    E2, _ = ex.enumerate_states_j(L, Jx2, Jy)
    assert np.all((E2 + 2 * 16 - o2.level_offset) % 4 == 0)
    with pytest.raises(Exception):
        o.set_couplings(np.zeros(16, dtype=np.int8), Jy)               # J must be +-1


@pytest.mark.parametrize("beta", [0.3, 0.8])
def test_sweep_with_couplings_samples_boltzmann_L4(beta):
    L, n = 4, 40000
    Jx, Jy = _random_j(L, 12)                                            # a frustrated sample
    rng = np.random.default_rng(7)
    sp = rng.integers(0, 2, (n, 16), dtype=np.uint8)
    po.sweep_slots_j(L, 13, 0, beta, 200, np.arange(n), sp, Jx, Jy)
    E, _ = po.energies_of_j(L, sp, Jx, Jy)
    exact = ex.exact_small_j(beta, L, Jx, Jy)
    chi2, dof = 0.0, 0
    for Ev, p in exact["pE"].items():
        if p * n < 5:
            continue
        chi2 += (int((E == Ev).sum()) - p * n) ** 2 / (p * n)
        dof += 1
    assert dof >= 4
    assert chi2 < dof + 6 * math.sqrt(2 * dof), (chi2, dof)


def test_pa_run_with_couplings_matches_enumeration_L4():
    # whole annealing runs on a frustrated sample with an ODD number of negative bonds (level offset 2): observables, free
    # energy, and the multi-histogram reweighting (Eq. 9 with E_m = -2N + 4m + e0) against the exact enumeration
    L, R, theta = 4, 3000, 5
    Jx, Jy = _random_j(L, 21)
    if ((Jx < 0).sum() + (Jy < 0).sum()) % 2 == 0:
        Jx[0] = -Jx[0]
    betas = [i / 25 for i in range(41)]                                  # 0 .. 1.6
    grid = np.array([0.1, 0.5, 1.1, 1.58])
    vals, rew = [], []
    for seed in range(500, 516):
        o = po.Oracle(L, R, seed); o.set_couplings(Jx, Jy)
        assert o.level_offset == 2
        vals.append(pa_driver.run_fixed(o, betas, theta, hist=True))
        rew.append({**o.reweight(grid), **o.reweight_mag(grid)})
    for i in (5, 15, 25, 40):
        exact = ex.exact_small_j(betas[i], L, Jx, Jy)
        for key in ("e", "C", "absm", "m2", "betaF_per_N", "S_per_N"):
            v = np.array([r[i][key] for r in vals])
            sigma = v.std(ddof=1) / math.sqrt(len(v))
            assert abs(v.mean() - exact[key]) < 4 * sigma + 1e-12, (betas[i], key, v.mean(), exact[key], sigma)
    for gi, b in enumerate(grid):
        exact = ex.exact_small_j(float(b), L, Jx, Jy)
        for key in ("lnZ", "e", "C", "absm", "m2"):
            v = np.array([r[key][gi] for r in rew])
            sigma = v.std(ddof=1) / math.sqrt(len(v))
            assert abs(v.mean() - exact[key]) < 4 * sigma + 1e-12, (b, key, v.mean(), exact[key], sigma)
