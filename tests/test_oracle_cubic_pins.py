"""Pins of the oracle's simple-cubic mode (O16; "models on different lattices in various dimensions",
L43 "3D Ising systems") against things other than itself (-m "not gpu"):

  energies ............ numpy.roll brute force on boxes with three different edges (a transposed axis fails), the closed-form
                        states (all up: -3N; 3D checkerboard: +3N, M = 0; planes), E = -3N (mod 4), the double bond of an edge of 2
  sweep ............... one whole sweep restated in numpy from explicit Philox counters on a 6 x 4 x 2 box (neighbour slots,
                        colour order, three thresholds); the exact Boltzmann distribution of the 4 x 2 x 2 box (2^16 states,
                        brute force) in chi^2 at three temperatures; global-flip symmetry; theta = 0
  whole method ........ PA runs on the 4 x 2 x 2 box against the enumeration for every observable of Eq. 3-5 (4 sigma over 16
                        seeds), sum ln Q against the enumeration's ln Z (Eq. 4), ln Omega(E) against the exact ln g(E) (Eq. 9)
  thresholds .......... closed forms
The enumeration (oracle/exact_ising.py::enumerate_box) is itself checked against the hand count of the 2 x 2 x 2 cube."""
import math

import numpy as np
import pytest

from oracle import exact_ising as ex
from oracle import pa_oracle as po
import pa_driver


def test_box_enumeration_against_hand_count_of_the_cube():
    # 2 x 2 x 2 with double bonds = the cube graph with J = 2: E = -24 + 4 k, k = number of cut edges.
    # k = 0: 2 states; one corner flipped cuts 3 edges: 8 x 2 = 16; two adjacent corners cut 4: 12 x 2, a face cuts 4: 3 x 2
    g = ex.density_of_states_box((2, 2, 2))
    assert g[-24] == 2 and g[-12] == 16 and g[-8] == 30 and sum(g.values()) == 256
    assert all(g[e] == g[-e] for e in g)                               # bipartite: flipping one sub-lattice maps E -> -E
    g = ex.density_of_states_box((4, 2, 2))
    assert sum(g.values()) == 65536 and g[-48] == 2 and g[48] == 2 and -44 not in g and -40 not in g
    # one flipped spin: 2 single bonds along x, 2 double bonds: 6 unsatisfied -> E = -48 + 12
    assert g[-36] == 2 * 16


def test_thresholds3_closed_forms():
    assert po.thresholds3(0.0) == (2**32 - 1,) * 3
    b = math.log(2.0) / 4                                              # exp(-4b) = 1/2, exp(-8b) = 1/4, exp(-12b) = 1/8
    t4, t8, t12 = po.thresholds3(b)
    assert abs(t4 - 2**31) <= 1 and abs(t8 - 2**30) <= 1 and abs(t12 - 2**29) <= 1
    assert po.thresholds3(0.3)[:2] == po.thresholds(0.3)


@pytest.mark.parametrize("dims", [(6, 4, 2), (4, 2, 2), (2, 2, 2), (8, 6, 4)])
def test_energies_3d_against_numpy_roll_and_closed_forms(dims):
    Lx, Ly, Lz = dims
    N = Lx * Ly * Lz
    rng = np.random.default_rng(1)
    sp = rng.integers(0, 2, (40, N), dtype=np.uint8)
    zz, yy, xx = np.meshgrid(np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    sp[0] = 1                                                          # all up
    sp[1] = ((xx + yy + zz) & 1).reshape(-1)                           # 3D checkerboard: every bond unsatisfied
    sp[2] = (zz & 1).reshape(-1)                                       # alternating planes: only the z bonds are unsatisfied
    sp[3] = (xx & 1).reshape(-1)
    E, M = po.energies_of_3d(dims, sp)
    g = sp.reshape(-1, Lz, Ly, Lx).astype(np.int64) * 2 - 1
    Eb = -(g * (np.roll(g, -1, 3) + np.roll(g, -1, 2) + np.roll(g, -1, 1))).sum((1, 2, 3))
    assert np.array_equal(E, Eb) and np.array_equal(M, g.sum((1, 2, 3)))
    assert E[0] == -3 * N and M[0] == N
    assert E[1] == 3 * N and M[1] == 0
    assert E[2] == -2 * N + N and E[3] == -2 * N + N and M[2] == 0    # two directions satisfied, one not
    assert np.all((E + 3 * N) % 4 == 0)
    # a single flipped spin in the all-up state breaks its six neighbour slots: E = -3N + 12 whatever the edges
    one = np.ones((1, N), dtype=np.uint8); one[0, N // 2 + 1] = 0
    assert po.energies_of_3d(dims, one)[0][0] == -3 * N + 12


def test_sweep_3d_counter_layout_and_acceptance_rule():
    """O16 restated in numpy on a box with three different edges: x(j,s,t,c) = philox(s, j>>2, 2t+c, 1)[j&3] with
    s = (z*Ly + y)*Lx + x, colour (x+y+z)&1 with colour 0 first, six neighbour slots (both slots of the edge of 2 count),
    flip iff u >= 3, or u = 2 and x < T4, or u = 1 and x < T8, or u = 0 and x < T12."""
    dims = (6, 4, 2)
    Lx, Ly, Lz = dims
    N = Lx * Ly * Lz
    beta, t, seed = 0.17, 77, (3 << 32) | 5
    key = [seed & 0xffffffff, seed >> 32]
    T = {d: min(math.floor(math.exp(-beta * d) * 2.0**32), 2**32 - 1) for d in (4, 8, 12)}
    assert (T[4], T[8], T[12]) == po.thresholds3(beta)
    slots = np.array([0, 3, 5, 31, 32, 4097, 2**31 - 1], dtype=np.int64)
    rng = np.random.default_rng(4)
    init = rng.integers(0, 2, (slots.size, N), dtype=np.uint8)
    init[0] = 1; init[1] = 0                                           # u = 0 everywhere at the start
    got = po.sweep_slots_3d(dims, seed, t, beta, 1, slots, init.copy())
    seen = set()
    for i, j in enumerate(int(v) for v in slots):
        sp = init[i].reshape(Lz, Ly, Lx).copy()
        for c in (0, 1):
            for z in range(Lz):
                for y in range(Ly):
                    for x in range(Lx):
                        if (x + y + z) & 1 != c:
                            continue
                        nb = [sp[z, y, (x - 1) % Lx], sp[z, y, (x + 1) % Lx], sp[z, (y - 1) % Ly, x], sp[z, (y + 1) % Ly, x],
                              sp[(z - 1) % Lz, y, x], sp[(z + 1) % Lz, y, x]]
                        u = sum(int(v != sp[z, y, x]) for v in nb)
                        xr = int(po.philox4x32_10([(z * Ly + y) * Lx + x, j >> 2, 2 * t + c, 1], key)[j & 3])
                        flip = u >= 3 or (u == 2 and xr < T[4]) or (u == 1 and xr < T[8]) or (u == 0 and xr < T[12])
                        seen.add((u, bool(flip)))
                        if flip:
                            sp[z, y, x] ^= 1
        assert np.array_equal(got[i].reshape(Lz, Ly, Lx), sp), j
    assert {(0, True), (0, False), (1, True), (1, False), (2, True), (2, False), (3, True), (4, True)} <= seen
    two = po.sweep_slots_3d(dims, seed, t, beta, 2, slots, init.copy())
    assert np.array_equal(two, po.sweep_slots_3d(dims, seed, t + 1, beta, 1, slots, got.copy()))


@pytest.mark.parametrize("beta", [0.1, 0.2216544, 0.4])
def test_sweep_3d_samples_boltzmann_4x2x2(beta):
    # 0.2216544 = the critical coupling of the infinite simple-cubic lattice (for orientation; the box has 16 spins)
    dims, n = (4, 2, 2), 40000
    rng = np.random.default_rng(6)
    sp = rng.integers(0, 2, (n, 16), dtype=np.uint8)
    po.sweep_slots_3d(dims, 9, 0, beta, 120, np.arange(n), sp)
    E, M = po.energies_of_3d(dims, sp)
    exact = ex.exact_box(beta, dims)
    chi2, dof = 0.0, 0
    for Ev, p in exact["pE"].items():
        if p * n < 5:
            continue
        cnt = int((E == Ev).sum())
        chi2 += (cnt - p * n) ** 2 / (p * n)
        dof += 1
    assert dof >= 5
    assert chi2 < dof + 6 * math.sqrt(2 * dof), (chi2, dof)
    assert abs(np.abs(M).mean() / 16 - exact["absm"]) < 5 * 0.5 / math.sqrt(n)
    assert abs(M.mean() / 16) < 5 / math.sqrt(n)


def test_sweep_3d_global_flip_symmetry_noop_and_slot_keying():
    dims, n = (4, 6, 2), 30
    N = 48
    rng = np.random.default_rng(2)
    a = rng.integers(0, 2, (n, N), dtype=np.uint8)
    b = (1 - a).copy(); a0 = a.copy()
    slots = np.arange(500, 500 + n)
    po.sweep_slots_3d(dims, 3, 9, 0.2, 0, slots, a)
    assert np.array_equal(a, a0)                                       # theta = 0
    po.sweep_slots_3d(dims, 3, 9, 0.2, 5, slots, a)
    po.sweep_slots_3d(dims, 3, 9, 0.2, 5, slots, b)
    assert np.array_equal(a, 1 - b) and not np.array_equal(a, a0)      # acceptance depends on u only
    perm = np.arange(n)[::-1].copy()
    c = po.sweep_slots_3d(dims, 3, 9, 0.2, 5, slots[perm], a0[perm].copy())
    assert np.array_equal(c, a[perm])                                  # keyed by slot, not by position in the call
    assert not np.array_equal(po.sweep_slots_3d(dims, 4, 9, 0.2, 5, slots, a0.copy()), a)


def test_box_oracle_init_and_beta0_closed_forms():
    dims, R = (6, 4, 4), 6000
    N = 96
    o = po.Oracle.box(dims, R, 8)
    assert o.N == N and o.nlev == 3 * N // 2 and o.population == R
    assert o.lnZ == pytest.approx(N * math.log(2.0), rel=1e-15)        # L93
    E, M = o.energies()
    assert abs(E.mean()) < 5 * math.sqrt(3 * N / R)                    # i.i.d. spins: <E> = 0, Var E = number of bonds = 3N
    assert abs(E.astype(float).var() / (3 * N) - 1) < 5 * math.sqrt(2 / R) * 1.5
    obs = o.observables(0.0)
    assert abs(obs["m2"] - 1 / N) < 5 * math.sqrt(2.0) / N / math.sqrt(R)
    assert obs["S_per_N"] == pytest.approx(math.log(2.0), rel=1e-12) and obs["betaF_per_N"] == pytest.approx(-math.log(2.0), rel=1e-12)
    # the INIT stream is keyed by (site, slot): the first replicas of a larger population are the same
    big = po.Oracle.box(dims, 2 * R, 8)
    assert np.array_equal(big.get_spins(0, 64), o.get_spins(0, 64))
    # modes that are 2D readings are refused
    with pytest.raises(RuntimeError):
        o.set_rng_mode(po.RNG_LCG)
    with pytest.raises(RuntimeError):
        o.set_couplings(np.ones(N, np.int8), np.ones(N, np.int8))


def test_pa_run_on_the_4x2x2_box_matches_enumeration():
    """The whole method on the simple-cubic box: every observable of Eq. 3-5 at five temperatures, sum_k ln Q_k against the
    enumeration's ln Z (Eq. 4: beta F / N), the population size bound (L69), and Eq. 9's ln Omega(E) against ln g(E)."""
    dims, R, theta = (4, 2, 2), 4000, 5
    N = 16
    betas = [i / 80 for i in range(41)]                                # 0 .. 0.5 (the box orders around 0.2)
    seeds = list(range(700, 716))
    runs, pops = [], []
    for s in seeds:
        o = po.Oracle.box(dims, R, s)
        runs.append(pa_driver.run_fixed(o, betas, theta, hist=True))
        pops.append(o)
    for i in (4, 12, 18, 26, 40):
        exact = ex.exact_box(betas[i], dims)
        for key in ("e", "C", "absm", "m2", "m4", "betaF_per_N", "S_per_N"):
            vals = np.array([r[i][key] for r in runs])
            sigma = vals.std(ddof=1) / math.sqrt(len(seeds))
            assert abs(vals.mean() - exact[key]) < 4 * sigma + 1e-12, (betas[i], key, vals.mean(), exact[key], sigma)
    for r in runs:
        assert all(abs(o["R"] - R) <= 4 * math.sqrt(R) / 2 * 1.5 for o in r)
    g = ex.density_of_states_box(dims)
    nlev = 3 * N // 2
    errs = []
    for o, r in zip(pops, runs):
        H, lnD = o.histogram()
        assert H.size == nlev + 1 and H.sum() == sum(x["R"] for x in r)     # L127
        E_of = -3 * N + 4 * np.arange(nlev + 1)
        SE = sum(round(x["e"] * x["R"] * N) for x in r)
        assert int((H * E_of).sum()) == SE
        for m in range(nlev + 1):
            if int(E_of[m]) not in g:
                assert H[m] == 0                                           # E = +-44, +-40 do not exist on this box
            elif E_of[m] <= 0:
                assert H[m] > 30
                errs.append((math.log(H[m]) - lnD[m]) - math.log(g[int(E_of[m])]))
    errs = np.array(errs).reshape(len(pops), -1)
    sig = errs.std(0, ddof=1) / math.sqrt(len(pops))
    assert np.all(np.abs(errs.mean(0)) < 4 * sig + 5e-3), (errs.mean(0), sig)
    # reweighting of the accumulated sums (O12) to an off-grid temperature, with e and C per SITE
    grid = np.array([0.03125, 0.21, 0.47])
    vals = {k: np.array([o.reweight(grid)[k] for o in pops]) for k in ("lnZ", "e", "C")}
    mags = {k: np.array([o.reweight_mag(grid)[k] for o in pops]) for k in ("absm", "m2")}
    for gi, b in enumerate(grid):
        exact = ex.exact_box(float(b), dims)
        for k, v in list(vals.items()) + list(mags.items()):
            col = v[:, gi]
            sigma = col.std(ddof=1) / math.sqrt(len(pops))
            assert abs(col.mean() - exact[k]) < 4 * sigma + 1e-12, (b, k, col.mean(), exact[k], sigma)
