"""Pins of the oracle's LCG-assisted sweep stream (O11; Sec. 4) against
what the paper and the mathematics fix (-m "not gpu").  None of the expected values comes from the
oracle itself or from the CUDA path."""
import math

import numpy as np
import pytest

from oracle import exact_ising as ex
from oracle import pa_oracle as po
import pa_driver

LCG = po.RNG_LCG


def test_lcg_recurrence_and_constants_of_the_paper():
    # r_{n+1} = A r_n + C mod 2^32 with A = 1664525 and C = 1013904223 (ref. [43]);
    # checked in unbounded integer arithmetic, including the wrap-around cases
    rng = np.random.default_rng(0)
    for r in [0, 1, 2**32 - 1, 2**31, 2**31 - 1] + [int(v) for v in rng.integers(0, 2**32, 200)]:
        assert po.lcg_next(r) == (1664525 * r + 1013904223) % 2**32
    # full period 2^32 (Hull-Dobell: C odd, A = 1 mod 4): r -> r' is a bijection, spot-checked on a block
    outs = {po.lcg_next(r) for r in range(5000)}
    assert len(outs) == 5000


@pytest.mark.parametrize("beta", [0.2, 0.4406868, 0.7])
def test_lcg_sweep_samples_boltzmann_L4(beta):
    # detailed balance: long fixed-beta chains against the exact Boltzmann distribution of the 4x4 torus
    L, n = 4, 40000
    rng = np.random.default_rng(6)
    sp = rng.integers(0, 2, (n, 16), dtype=np.uint8)
    po.sweep_slots(L, seed=10, t0=0, beta=beta, theta=150, slot_ids=np.arange(n), spins01=sp, rng_mode=LCG)
    E, M = po.energies_of(L, sp)
    exact = ex.exact_small(beta, L)
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


def test_lcg_sweep_symmetry_noop_and_keying():
    L, n = 6, 70                                                       # 70 slots: three words, the last one ragged
    rng = np.random.default_rng(1)
    a = rng.integers(0, 2, (n, L * L), dtype=np.uint8)
    b = (1 - a).copy()
    a0 = a.copy()
    slots = np.arange(100, 100 + n)
    po.sweep_slots(L, 3, 17, 0.35, 0, slots, a, rng_mode=LCG)
    assert np.array_equal(a, a0)                                       # theta = 0 is a no-op
    po.sweep_slots(L, 3, 17, 0.35, 7, slots, a, rng_mode=LCG)
    po.sweep_slots(L, 3, 17, 0.35, 7, slots, b, rng_mode=LCG)
    assert np.array_equal(a, 1 - b)                                    # global flip symmetry (acceptance depends on u only)
    assert not np.array_equal(a, a0)
    # theta = 3 split into 1 + 2 with the counter advanced: the word is re-seeded at every visit (O11)
    base = rng.integers(0, 2, (n, L * L), dtype=np.uint8)
    ref = po.sweep_slots(L, 3, 5, 0.4, 3, slots, base.copy(), rng_mode=LCG)
    s = po.sweep_slots(L, 3, 5, 0.4, 1, slots, base.copy(), rng_mode=LCG)
    s = po.sweep_slots(L, 3, 6, 0.4, 2, slots, s, rng_mode=LCG)
    assert np.array_equal(s, ref)
    # a replica's trajectory depends on its slot id, not on its position in the call
    perm = np.arange(n)[::-1].copy()
    s = po.sweep_slots(L, 3, 5, 0.4, 3, slots[perm], base[perm].copy(), rng_mode=LCG)
    assert np.array_equal(s, ref[perm])
    # other seed / counter / slot / generator mode -> other trajectory
    assert not np.array_equal(po.sweep_slots(L, 4, 5, 0.4, 3, slots, base.copy(), rng_mode=LCG), ref)
    assert not np.array_equal(po.sweep_slots(L, 3, 6, 0.4, 3, slots, base.copy(), rng_mode=LCG), ref)
    assert not np.array_equal(po.sweep_slots(L, 3, 5, 0.4, 3, slots + 1, base.copy(), rng_mode=LCG), ref)
    assert not np.array_equal(po.sweep_slots(L, 3, 5, 0.4, 3, slots, base.copy()), ref)


def test_lcg_siblings_in_one_word_decorrelate():
    # with ONE random number per word, copies of the same parent stored in the same word
    # "are coupled and remain identical for all future times"; the LCG gives every replica of the word its own
    # number (L236), so identical copies in one word must drift apart
    L = 8
    rng = np.random.default_rng(3)
    one = rng.integers(0, 2, (1, L * L), dtype=np.uint8)
    sp = np.repeat(one, 32, axis=0).copy()                             # 32 identical replicas = one full word
    po.sweep_slots(L, 7, 0, 0.3, 2, np.arange(32), sp, rng_mode=LCG)
    distinct = {row.tobytes() for row in sp}
    assert len(distinct) == 32
    # and their mutual overlap is that of independent chains: mean Hamming distance between siblings is the same
    # as between the same configuration evolved in different words (statistically, 5 sigma)
    n = 256
    same_word = np.repeat(one, n, axis=0).copy()
    po.sweep_slots(L, 7, 0, 0.3, 2, np.arange(n), same_word, rng_mode=LCG)
    other_words = np.repeat(one, n, axis=0).copy()
    po.sweep_slots(L, 7, 0, 0.3, 2, np.arange(n) * 32, other_words, rng_mode=LCG)
    d_same = np.array([(same_word[i] != same_word[i + 1]).sum() for i in range(0, n, 2) if (i // 32) == ((i + 1) // 32)])
    d_other = np.array([(other_words[i] != other_words[i + 1]).sum() for i in range(0, n, 2)])
    se = math.sqrt(d_same.var(ddof=1) / d_same.size + d_other.var(ddof=1) / d_other.size)
    assert abs(d_same.mean() - d_other.mean()) < 5 * se, (d_same.mean(), d_other.mean(), se)


def _runs(L, R, betas, theta, seeds, mode):
    out = []
    for s in seeds:
        o = po.Oracle(L, R, s)
        o.set_rng_mode(mode)
        out.append(pa_driver.run_fixed(o, betas, theta))
    return out


def test_lcg_pa_run_matches_exact_enumeration_L4():
    L, R, theta = 4, 4000, 5
    betas = [i / 40 for i in range(41)]
    seeds = list(range(200, 216))
    runs = _runs(L, R, betas, theta, seeds, LCG)
    for i in (4, 12, 18, 24, 40):
        exact = ex.exact_small(betas[i], L)
        for key in ("e", "C", "absm", "m2", "m4", "betaF_per_N", "S_per_N"):
            vals = np.array([r[i][key] for r in runs])
            sigma = vals.std(ddof=1) / math.sqrt(len(seeds))
            assert abs(vals.mean() - exact[key]) < 4 * sigma + 1e-12, (betas[i], key, vals.mean(), exact[key], sigma)


def test_lcg_pa_run_matches_kaufman_and_variance_ratio_L16(cfg1_oracle_runs):
    # configs[0] of BASELINE.json (L=16, R=1000, 100 steps, theta=10) with the LCG-assisted stream: exact finite-L
    # results (Kaufman) within the seed scatter, and Table 1's last column (L201-L204): the variance of C is the
    # same as with one Philox number per spin (ratio 1; here 16 + 16 seeds, the Philox runs are the session's shared ones)
    L, R, theta = 16, 1000, 10
    betas, shared = cfg1_oracle_runs
    lcg = _runs(L, R, betas, theta, list(range(21, 37)), LCG)
    phi = [obs for _, obs in shared]
    for i in (10, 30, 44, 60, 100):
        k = ex.kaufman(betas[i], L)
        for key in ("e", "C", "betaF_per_N", "S_per_N"):
            vals = np.array([r[i][key] for r in lcg])
            sigma = vals.std(ddof=1) / math.sqrt(len(lcg))
            assert abs(vals.mean() - k[key]) < 4 * sigma + 1e-9, (betas[i], key, vals.mean(), k[key], sigma)
    ratios = []
    for i in range(40, 101, 4):                                        # the critical and low-temperature range of Fig. 2(c)
        v1 = np.var([r[i]["C"] for r in lcg], ddof=1)
        v0 = np.var([r[i]["C"] for r in phi], ddof=1)
        ratios.append(v1 / v0)
    gm = math.exp(np.mean(np.log(ratios)))                             # geometric mean over 16 temperatures
    assert 0.4 < gm < 2.5, (gm, ratios)                                # n_RNG = 1 without the LCG would give ~32 (Table 1)


def _lcg_seed_counter(L, x, y, g, t, c):
    """The (Philox counter, output word) that seeds the word of group g at site (x, y) at its visit (sweep t, colour c): O11 as
    include/pa.h publishes it, written out here independently of the oracle."""
    return ((y >> 2) * (L // 2) + (x >> 1), g, 2 * t + c, 3), y & 3


@pytest.mark.parametrize("L", [8, 12])
def test_lcg_stream_seed_and_lane_layout_from_explicit_counters(L):
    """O11 (Sec. 4) with the layout written out: the word of group g = j >> 5 at site (x, y) is seeded at
    every visit (sweep t, colour c = (x + y) & 1) by r_0 = philox((y >> 2)(L/2) + (x >> 1), g, 2t + c, TAG_LCG = 3)[y & 3] with key
    (seed & 2^32-1, seed >> 32), and replica j takes x_j = r_{32 - (j & 31)} of r_{n+1} = 1664525 r_n + 1013904223 mod 2^32
    (most significant lane first).  One whole sweep of replicas in several words is recomputed site by site from explicit Philox
    counters (the Philox routine itself is pinned against cuRAND's header in test_oracle_pins.py) and Python-integer LCG steps:
    colour-0 decisions from the initial state, colour-1 decisions from the updated colour-0 neighbours.  L = 8 and 12 so that the
    quad row y >> 2 takes two and three values (the chi-square pin at L = 4 cannot see a quad index that collides between rows);
    a wrong output word, tag, jump length, lane order or counter slot fails here.  All branches of the acceptance rule occur."""
    beta, t = 0.33, 4321
    N = L * L
    seed = (5 << 32) | 777                                             # both key words in use
    key = [seed & 0xffffffff, seed >> 32]
    T4 = min(math.floor(math.exp(-4 * beta) * 2.0**32), 2**32 - 1)
    T8 = min(math.floor(math.exp(-8 * beta) * 2.0**32), 2**32 - 1)
    slots = np.array([0, 1, 2, 30, 31, 32, 33, 63, 64, 1000003, 2**31 - 5], dtype=np.int64)
    rng = np.random.default_rng(4)
    init = rng.integers(0, 2, (slots.size, N), dtype=np.uint8)
    got = po.sweep_slots(L, seed, t, beta, 1, slots, init.copy(), rng_mode=LCG)
    seen = set()
    for i, j in enumerate(int(v) for v in slots):
        sp = init[i].reshape(L, L).copy()
        for c in (0, 1):
            for y in range(L):
                for x in range(L):
                    if (x + y) & 1 != c:
                        continue
                    ctr, word = _lcg_seed_counter(L, x, y, j >> 5, t, c)
                    r = int(po.philox4x32_10(list(ctr), key)[word])
                    for _ in range(32 - (j & 31)):
                        r = (1664525 * r + 1013904223) % 2**32
                    nb = [sp[y, (x - 1) % L], sp[y, (x + 1) % L], sp[(y - 1) % L, x], sp[(y + 1) % L, x]]
                    u = sum(int(v != sp[y, x]) for v in nb)
                    flip = u >= 2 or (u == 1 and r < T4) or (u == 0 and r < T8)
                    seen.add((u, bool(flip)))
                    if flip:
                        sp[y, x] ^= 1
        assert np.array_equal(got[i].reshape(L, L), sp), j
    assert {(0, True), (0, False), (1, True), (1, False), (2, True)} <= seen
    # the sweep counter advances by one per sweep, as in the Philox stream
    two = po.sweep_slots(L, seed, t, beta, 2, slots, init.copy(), rng_mode=LCG)
    assert np.array_equal(two, po.sweep_slots(L, seed, t + 1, beta, 1, slots, got.copy(), rng_mode=LCG))


def test_lcg_seeds_of_distinct_words_and_visits_are_distinct_draws():
    """O11: no two (word, visit) pairs share a seed draw.  Over every site of an L = 16 lattice x 3 groups x 2 sweeps (the colour
    follows from the site) the (counter, output word) pairs are pairwise distinct -- in particular the quad index separates
    the rows 0-3, 4-7, ... and the two columns of a pair x >> 1 are told apart by their colour in the third counter word --
    and, Philox being a bijection of the counter, the r_0 actually drawn are distinct 32-bit words of distinct 128-bit blocks:
    checked on the values too (a birthday collision among 1536 uniform 32-bit words has probability 3e-4)."""
    L = 16
    draws, values = set(), []
    key = [2024, 9]
    for t in (0, 1):
        for g in (0, 1, 5):
            for y in range(L):
                for x in range(L):
                    ctr, word = _lcg_seed_counter(L, x, y, g, t, (x + y) & 1)
                    assert (ctr, word) not in draws, (x, y, g, t)
                    draws.add((ctr, word))
                    values.append(int(po.philox4x32_10(list(ctr), key)[word]))
    assert len(draws) == 2 * 3 * L * L
    assert len(set(values)) == len(values)
    # every quad counter stays inside [0, (L/4)(L/2)) and every (quad, output word, colour) is used exactly once per (g, t)
    quads = {c[0][0] for c in draws}
    assert quads == set(range((L // 4) * (L // 2)))
