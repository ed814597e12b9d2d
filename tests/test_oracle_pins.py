"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

Each test names the oracle function it pins and the passage / closed form it is pinned to.
None of the expected values comes from the oracle itself or from the CUDA path.
"""
import ctypes as C
import math
import os
import subprocess

import numpy as np
import pytest

from oracle import exact_ising as ex
from oracle import pa_oracle as po
import pa_driver

HERE = os.path.dirname(os.path.abspath(__file__))


# ---------------------------------------------------------------------------------------------
# O1 Philox4x32-10  <-  cuRAND's own header ("included as one of the generators in
# the curand library"), compiled for the host: an implementation independent of the oracle's.
# ---------------------------------------------------------------------------------------------

@pytest.fixture(scope="module")
def curand_ref(tmp_path_factory):
    cuda_inc = "/usr/local/cuda/include"
    if not os.path.exists(os.path.join(cuda_inc, "curand_philox4x32_x.h")):
        pytest.skip("CUDA toolkit headers not present")
    so = str(tmp_path_factory.mktemp("curand") / "libcurand_ref.so")
    subprocess.run(["g++", "-O1", "-fPIC", "-shared", "-I", cuda_inc, "-o", so,
                    os.path.join(HERE, "helpers", "curand_philox_ref.cpp")], check=True)
    lib = C.CDLL(so)
    lib.curand_ref_philox.argtypes = [C.c_void_p] * 3
    lib.curand_ref_philox.restype = None

    def f(ctr, key):
        ctr = np.ascontiguousarray(ctr, dtype=np.uint32); key = np.ascontiguousarray(key, dtype=np.uint32)
        out = np.empty(4, dtype=np.uint32)
        lib.curand_ref_philox(ctr.ctypes.data, key.ctypes.data, out.ctypes.data)
        return out
    return f


def test_philox_matches_curand_header(curand_ref):
    rng = np.random.default_rng(12345)
    cases = [([0, 0, 0, 0], [0, 0]), ([0xffffffff] * 4, [0xffffffff] * 2), ([1, 2, 3, 4], [5, 6])]
    cases += [(rng.integers(0, 2**32, 4, dtype=np.uint64), rng.integers(0, 2**32, 2, dtype=np.uint64))
              for _ in range(2000)]
    for ctr, key in cases:
        assert np.array_equal(po.philox4x32_10(ctr, key), curand_ref(ctr, key)), (ctr, key)


def test_philox_is_injective_on_a_counter_block():
    # a bijection of the counter for a fixed key: distinct counters -> distinct 128-bit outputs
    seen = set()
    for c0 in range(64):
        for c1 in range(64):
            seen.add(tuple(po.philox4x32_10([c0, c1, 7, 1], [1, 0]).tolist()))
    assert len(seen) == 64 * 64


def test_philox_output_words_are_uniform_bits():
    # each of the 128 output bits is set about half of the time (catches a dropped round / word)
    n = 4096
    acc = np.zeros(128)
    for i in range(n):
        o = po.philox4x32_10([i, 0, 0, 1], [3, 0])
        acc += np.unpackbits(o.view(np.uint8))
    assert np.all(np.abs(acc / n - 0.5) < 5 * 0.5 / math.sqrt(n))


# ---------------------------------------------------------------------------------------------
# O2 thresholds  <-  closed forms
# ---------------------------------------------------------------------------------------------

def test_thresholds_closed_forms():
    assert po.threshold(1.0) == 2**32 - 1            # beta = 0: accept with 1 - 2^-32
    assert po.threshold(0.5) == 2**31
    assert po.threshold(2.0**-32) == 1
    assert po.threshold(0.0) == 0
    assert po.threshold(0.75) == 3 * 2**30
    for beta in (0.01, 0.2, 0.4406868, 1.0, 3.0):
        t4, t8 = po.thresholds(beta)
        assert t8 <= t4
        assert t4 == int(math.floor(math.exp(-4 * beta) * 2**32))
        assert t8 == int(math.floor(math.exp(-8 * beta) * 2**32))
        # exp(-8b) = exp(-4b)^2 (Metropolis factor of dE = 8 is the square of that of dE = 4)
        assert abs(t8 / 2**32 - (t4 / 2**32) ** 2) < 2e-9


# ---------------------------------------------------------------------------------------------
# O4 energies  <-  brute force (numpy.roll), special states
# ---------------------------------------------------------------------------------------------

def _brute_energy(sp01, L):
    g = sp01.reshape(-1, L, L).astype(np.int64) * 2 - 1
    E = -(g * np.roll(g, -1, 2)).sum((1, 2)) - (g * np.roll(g, -1, 1)).sum((1, 2))
    return E.astype(np.int32), g.sum((1, 2)).astype(np.int32)


@pytest.mark.parametrize("L", [4, 6, 16])
def test_energies_bruteforce(L):
    rng = np.random.default_rng(L)
    sp = rng.integers(0, 2, (37, L * L), dtype=np.uint8)
    E, M = po.energies_of(L, sp)
    Eb, Mb = _brute_energy(sp, L)
    assert np.array_equal(E, Eb) and np.array_equal(M, Mb)
    assert np.all((E + 2 * L * L) % 4 == 0)                     # E = -2N + 4m on the even torus


def test_energies_special_states():
    L, N = 8, 64
    up = np.ones((1, N), dtype=np.uint8)
    yy, xx = np.divmod(np.arange(N), L)
    cb = (((xx + yy) & 1)[None, :]).astype(np.uint8)
    stripes = ((yy & 1)[None, :]).astype(np.uint8)              # rows alternate: vertical bonds broken
    E, M = po.energies_of(L, np.concatenate([up, 1 - up, cb, stripes]))
    assert E.tolist() == [-2 * N, -2 * N, 2 * N, 0]
    assert M.tolist() == [N, -N, 0, 0]


def test_energies_against_L4_enumeration():
    E_all, M_all = ex.enumerate_states(4)
    idx = np.arange(0, 65536, 17)
    sp = ((idx[:, None] >> np.arange(16)[None, :]) & 1).astype(np.uint8)
    E, M = po.energies_of(4, sp)
    assert np.array_equal(E, E_all[idx]) and np.array_equal(M, M_all[idx])


# ---------------------------------------------------------------------------------------------
# a0 init  <-  closed forms at beta = 0 (i.i.d. spins): <E>=0, Var E = 2N, <m^2> = 1/N,
# <m^4> = 3/N^2 - 2/N^3, S/N = ln 2, beta F / N = -ln 2
# ---------------------------------------------------------------------------------------------

def test_init_closed_forms():
    L, R = 8, 40000
    N = L * L
    o = po.Oracle(L, R, 77)
    E, M = o.energies()
    obs = o.observables(0.0)
    assert abs(E.mean()) < 5 * math.sqrt(2 * N / R)
    assert abs(E.var() / (2 * N) - 1) < 5 * math.sqrt(2 / R) * 1.5
    assert abs(obs["m2"] - 1 / N) < 5 * math.sqrt(2.0) / N / math.sqrt(R)
    assert abs(obs["m4"] - (3 / N**2 - 2 / N**3)) < 0.05 * 3 / N**2
    assert abs(M.mean()) < 5 * math.sqrt(N / R)
    assert obs["S_per_N"] == pytest.approx(math.log(2) + 0.0 * obs["e"], abs=1e-15)
    assert obs["betaF_per_N"] == pytest.approx(-math.log(2), abs=1e-15)
    assert obs["R"] == R and obs["lnQ"] == 0.0
    # every site and every replica is unbiased
    sp = o.get_spins()
    assert np.all(np.abs(sp.mean(0)) < 5 / math.sqrt(R))
    assert abs(sp.mean(1)).max() < 6 / math.sqrt(N)
    # two different seeds and two different replicas differ
    o2 = po.Oracle(L, 64, 78)
    assert not np.array_equal(o2.get_spins(), sp[:64])
    assert len({r.tobytes() for r in sp[:2000]}) == 2000


def test_init_stream_counter_layout():
    """O1 with the INIT counter layout written out: the word of (site s, group g) is philox(s, g >> 2, 0, TAG_INIT = 0)[g & 3] with key
    (seed & 2^32-1, seed >> 32); replica j is bit j & 31 of group j >> 5, a set bit is an up spin.  The statistics of
    test_init_closed_forms cannot see a wrong tag, a transposed counter or a reversed lane order; this recomputation can (the Philox
    routine itself is pinned against cuRAND's header above).  Square lattice and a box (site s = (z Ly + y) Lx + x, O16)."""
    seed = (11 << 32) | 12345                                          # both key words in use
    key = [seed & 0xffffffff, seed >> 32]
    for make, N, R in ((lambda: po.Oracle(6, 100, seed), 36, 100), (lambda: po.Oracle.box((4, 6, 2), 70, seed), 48, 70)):
        sp = make().get_spins()
        assert sp.shape == (R, N)
        for j in (0, 1, 31, 32, 33, 63, 64, R - 1):
            g, b = j >> 5, j & 31
            want = [1 if (int(po.philox4x32_10([s, g >> 2, 0, 0], key)[g & 3]) >> b) & 1 else -1 for s in range(N)]
            assert sp[j].tolist() == want, j


# ---------------------------------------------------------------------------------------------
# O3 sweep  <-  L = 4 brute force Boltzmann distribution, symmetries, no-op
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("beta", [0.2, 0.4406868, 0.7])
def test_sweep_samples_boltzmann_L4(beta):
    L, n = 4, 40000
    rng = np.random.default_rng(5)
    sp = rng.integers(0, 2, (n, 16), dtype=np.uint8)
    po.sweep_slots(L, seed=9, t0=0, beta=beta, theta=150, slot_ids=np.arange(n), spins01=sp)
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
    assert abs(M.mean() / 16) < 5 / math.sqrt(n) * 1.0


def test_sweep_stream_counter_layout_and_acceptance_rule():
    """O1 / O3 with the counter layout written out: x(j, s, t, c) = philox(s, j>>2, 2t+c, TAG_SWEEP=1)[j&3] with key
    (seed & 2^32-1, seed >> 32), colour 0 = (x+y) even first, flip iff u >= 2, or u = 1 and x < T4, or u = 0 and x < T8 with
    T = floor(exp(-beta dE) 2^32) (O2).  One whole sweep of random replicas is recomputed site by site in numpy from the
    explicit Philox counters (the Philox routine itself is pinned against cuRAND's header above): colour-0 decisions from the
    initial state, colour-1 decisions from the updated colour-0 neighbours.  All three branches of the rule occur."""
    L, beta, t = 6, 0.31, 12345
    N = L * L
    seed = (7 << 32) | 99                                              # both key words in use
    key = [seed & 0xffffffff, seed >> 32]
    T4 = min(math.floor(math.exp(-4 * beta) * 2.0**32), 2**32 - 1)
    T8 = min(math.floor(math.exp(-8 * beta) * 2.0**32), 2**32 - 1)
    assert (T4, T8) == po.thresholds(beta)
    slots = np.array([0, 1, 2, 3, 4, 31, 32, 33, 1000003, 2**31 - 5], dtype=np.int64)
    rng = np.random.default_rng(2)
    init = rng.integers(0, 2, (slots.size, N), dtype=np.uint8)
    got = po.sweep_slots(L, seed, t, beta, 1, slots, init.copy())
    seen = set()
    for i, j in enumerate(int(v) for v in slots):
        sp = init[i].reshape(L, L).copy()
        for c in (0, 1):
            for y in range(L):
                for x in range(L):
                    if (x + y) & 1 != c:
                        continue
                    nb = [sp[y, (x - 1) % L], sp[y, (x + 1) % L], sp[(y - 1) % L, x], sp[(y + 1) % L, x]]
                    u = sum(int(v != sp[y, x]) for v in nb)
                    xr = int(po.philox4x32_10([y * L + x, j >> 2, 2 * t + c, 1], key)[j & 3])
                    flip = u >= 2 or (u == 1 and xr < T4) or (u == 0 and xr < T8)
                    seen.add((u, bool(flip)))
                    if flip:
                        sp[y, x] ^= 1
        assert np.array_equal(got[i].reshape(L, L), sp), j
    assert {(0, True), (0, False), (1, True), (1, False), (2, True)} <= seen
    # the sweep counter advances by one per sweep: theta = 2 from t equals two calls at t and t + 1
    two = po.sweep_slots(L, seed, t, beta, 2, slots, init.copy())
    assert np.array_equal(two, po.sweep_slots(L, seed, t + 1, beta, 1, slots, got.copy()))


def test_sweep_siblings_in_one_quad_and_one_word_decorrelate():
    """Sibling replicas (copies of one parent, adjacent slots after resampling) share a Philox CALL when they sit in one quad
    4q..4q+3 (they take different output words of it) and a machine word when they sit in 32g..32g+31.  Every spin still has
    its own number (north_star's key tuple; Table 1's variance ratio 1, L193-L196), so identical copies must drift apart, and
    as fast as copies placed in different quads / words (PAPER.md L206-L208 is what goes wrong otherwise)."""
    L, beta, n = 8, 0.3, 512
    rng = np.random.default_rng(3)
    one = rng.integers(0, 2, (1, L * L), dtype=np.uint8)
    quad = np.repeat(one, 4, axis=0).copy()
    po.sweep_slots(L, 7, 0, beta, 2, np.arange(40, 44), quad)
    assert len({r.tobytes() for r in quad}) == 4
    word = np.repeat(one, 32, axis=0).copy()
    po.sweep_slots(L, 7, 0, beta, 2, np.arange(64, 96), word)
    assert len({r.tobytes() for r in word}) == 32
    adjacent = np.repeat(one, n, axis=0).copy()
    po.sweep_slots(L, 7, 0, beta, 2, np.arange(n), adjacent)
    apart = np.repeat(one, n, axis=0).copy()
    po.sweep_slots(L, 7, 0, beta, 2, np.arange(n) * 32, apart)         # every copy in a word (and quad) of its own
    d_quad = np.array([(adjacent[i] != adjacent[i + 1]).sum() for i in range(0, n, 2)])          # pairs inside one quad
    d_word = np.array([(adjacent[i] != adjacent[i + 5]).sum() for i in range(0, n - 8, 32)] +
                      [(adjacent[i + 2] != adjacent[i + 27]).sum() for i in range(0, n - 32, 32)])  # same word, different quads
    d_apart = np.array([(apart[i] != apart[i + 1]).sum() for i in range(0, n, 2)])
    for d in (d_quad, d_word):
        se = math.sqrt(d.var(ddof=1) / d.size + d_apart.var(ddof=1) / d_apart.size)
        assert abs(d.mean() - d_apart.mean()) < 4 * se, (d.mean(), d_apart.mean(), se)
    assert d_apart.mean() > 5                                          # they do move at beta = 0.3


def test_sweep_global_flip_symmetry_and_noop():
    # acceptance depends only on u (the number of anti-parallel neighbours): inverting every
    # spin gives the inverted trajectory, the same energies and opposite magnetisations
    L, n = 6, 50
    rng = np.random.default_rng(1)
    a = rng.integers(0, 2, (n, L * L), dtype=np.uint8)
    b = (1 - a).copy()
    a0 = a.copy()
    slots = np.arange(100, 100 + n)
    po.sweep_slots(L, 3, 17, 0.35, 0, slots, a)
    assert np.array_equal(a, a0)                                   # theta = 0 is a no-op
    po.sweep_slots(L, 3, 17, 0.35, 7, slots, a)
    po.sweep_slots(L, 3, 17, 0.35, 7, slots, b)
    assert np.array_equal(a, 1 - b)
    assert not np.array_equal(a, a0)


def test_sweep_depends_on_slot_sweep_counter_and_seed_only():
    L, n = 6, 8
    rng = np.random.default_rng(2)
    base = rng.integers(0, 2, (n, L * L), dtype=np.uint8)
    ref = po.sweep_slots(L, 3, 5, 0.4, 3, np.arange(n), base.copy())
    # splitting theta = 3 into 1 + 2 with the counter advanced gives the same trajectory
    s = po.sweep_slots(L, 3, 5, 0.4, 1, np.arange(n), base.copy())
    s = po.sweep_slots(L, 3, 6, 0.4, 2, np.arange(n), s)
    assert np.array_equal(s, ref)
    # a replica's trajectory depends on its slot id, not on its position in the call
    perm = np.arange(n)[::-1].copy()
    s = po.sweep_slots(L, 3, 5, 0.4, 3, perm, base[perm].copy())
    assert np.array_equal(s, ref[perm])
    # other seed / other counter / other slot -> other trajectory
    assert not np.array_equal(po.sweep_slots(L, 4, 5, 0.4, 3, np.arange(n), base.copy()), ref)
    assert not np.array_equal(po.sweep_slots(L, 3, 6, 0.4, 3, np.arange(n), base.copy()), ref)
    assert not np.array_equal(po.sweep_slots(L, 3, 5, 0.4, 3, np.arange(n) + 1, base.copy()), ref)


def test_sweep_ground_state_is_stable_at_low_T_and_melts_at_beta0():
    L = 8
    up = np.ones((4, L * L), dtype=np.uint8)
    cold = po.sweep_slots(L, 1, 0, 5.0, 5, np.arange(4), up.copy())   # exp(-8*5) ~ 4e-18
    assert np.array_equal(cold, up)
    hot = po.sweep_slots(L, 1, 0, 0.0, 1, np.arange(4), up.copy())    # T = 2^32-1: every spin flips
    assert np.array_equal(hot, 1 - up)


# ---------------------------------------------------------------------------------------------
# O5 TREE1024, W, lnQ  <-  exact arithmetic cases, math.fsum, histogram regrouping, dbeta = 0
# ---------------------------------------------------------------------------------------------

def test_tree1024_exact_cases():
    assert po.tree1024(np.zeros(0)) == 0.0
    for n in (1, 31, 32, 33, 1023, 1024, 1025, 5000):
        assert po.tree1024(np.ones(n)) == float(n)
        a = np.arange(1, n + 1, dtype=np.float64)
        assert po.tree1024(a) == n * (n + 1) / 2                     # integers: any order is exact
    rng = np.random.default_rng(0)
    a = rng.random(70001)
    assert po.tree1024(a) == pytest.approx(math.fsum(a), rel=1e-13)
    # the order is the stated one: pairwise inside a run of 32 (i, i+16), ... not left-to-right
    v = np.zeros(32); v[0] = 1.0; v[16] = 2.0**-53; v[1] = 2.0**-53
    # tree: (v0+v16) = 1 (ties-to-even), (v1+v17) = 2^-53, ... then 1 + 2^-53 -> 1.0
    assert po.tree1024(v) == 1.0
    v = np.zeros(32); v[16] = 2.0**-53; v[1] = 2.0**-53; v[17] = 0.0; v[0] = 1.0; v[8] = 0
    w = v.copy(); w[1] = 0; w[16] = 2.0**-52
    assert po.tree1024(w) == 1.0 + 2.0**-52


def test_weights_closed_forms_and_histogram_regrouping():
    rng = np.random.default_rng(3)
    N = 256
    E = (-2 * N + 4 * rng.integers(40, 200, 3000)).astype(np.int32)
    p0 = po.resample_plan(3000, E, seed=1, k=0, dbeta=0.0)
    assert p0["W"] == 3000.0 and p0["lnQ"] == 0.0                  # w = 1, Q = 1
    assert np.all(p0["r"] == 1) and p0["R_new"] == 3000           # tau_hat = 1 exactly: identity
    assert np.array_equal(p0["o"], np.arange(3000))
    db = 0.013
    p = po.resample_plan(3000, E, seed=1, k=0, dbeta=db)
    Eref = int(E.min())
    assert np.allclose(p["w"], np.exp(-db * (E - Eref)), rtol=1e-15, atol=0)
    vals, cnt = np.unique(E, return_counts=True)
    W_hist = math.fsum(c * math.exp(-db * (v - Eref)) for v, c in zip(vals, cnt))
    assert p["W"] == pytest.approx(W_hist, rel=1e-12)
    # Eq. 1 (L58): Q = (1/R) sum exp(-dbeta E_j), evaluated without the shift in high precision
    import mpmath as mp
    Q = mp.fsum(mp.exp(-mp.mpf(db) * int(e)) for e in E) / 3000
    assert p["lnQ"] == pytest.approx(float(mp.log(Q)), rel=1e-12)


# ---------------------------------------------------------------------------------------------
# O6/O7 copy numbers, scan, copy  <-  Eq. 2 (L67), L69, definitions
# ---------------------------------------------------------------------------------------------

def test_copy_numbers_eq2_properties():
    rng = np.random.default_rng(4)
    N = 1024
    R_target = 5000
    E = (-2 * N + 4 * rng.integers(100, 400, 4700)).astype(np.int32)      # R_cur != R_target
    db = 0.004
    p = po.resample_plan(R_target, E, seed=11, k=3, dbeta=db)
    tau = R_target * p["w"] / p["W"]
    assert tau.sum() == pytest.approx(R_target, rel=1e-12)                   # L69
    fl = np.floor(tau)
    assert np.all((p["r"] == fl) | (p["r"] == fl + 1))                       # Eq. 2
    assert np.array_equal(p["o"], np.concatenate([[0], np.cumsum(p["r"])[:-1]]))
    assert p["R_new"] == int(p["r"].sum())
    assert abs(p["R_new"] - R_target) <= 4 * math.sqrt(len(E)) / 2          # L69 "very small fluctuations"
    # the rounding is the stated Bernoulli: P(r = floor+1) = frac(tau); average over resample counters
    up = np.zeros(len(E))
    K = 400
    for k in range(K):
        up += po.resample_plan(R_target, E, seed=11, k=k, dbeta=db)["r"] - fl
    frac = tau - fl
    z = (up / K - frac) / np.sqrt(np.maximum(frac * (1 - frac), 1e-4) / K)
    assert np.abs(z).max() < 5.5 and abs(z.mean()) < 0.1
    # the uniform number of replica j at counter k is philox(j>>2, 0, k, TAG=2)[j&3] * 2^-32
    j, k = 1234, 3
    x = int(po.philox4x32_10([j >> 2, 0, k, 2], [11, 0])[j & 3])
    assert p["r"][j] == int(fl[j]) + (1 if x * 2.0**-32 < frac[j] else 0)


def test_resample_copies_parents_in_order():
    L, R = 6, 700
    o = po.Oracle(L, R, 5)
    o.sweep(0.3, 2)
    before = o.get_spins()
    E_before, _ = o.energies()
    R_new = o.resample(0.3, 0.45)
    dbg = o.resample_debug(R)
    after = o.get_spins()
    assert R_new == o.population == int(dbg["r"].sum())
    parent = np.repeat(np.arange(R), dbg["r"])                       # new[o_j + c] = old[j]
    assert np.all(np.diff(parent) >= 0)
    assert np.array_equal(after, before[parent])
    assert o.resample_counter == 1
    plan = po.resample_plan(R, E_before, 5, 0, 0.45 - 0.3)
    assert np.array_equal(plan["r"], dbg["r"]) and plan["W"] == dbg["W"]
    assert o.lnZ == pytest.approx(36 * math.log(2) + plan["lnQ"], rel=1e-15)


def test_resample_rejects_bad_arguments_and_capacity():
    o = po.Oracle(4, 64, 1)
    rc, _ = o.resample_rc(0.5, 0.4)
    assert rc != 0                                                   # beta' < beta
    assert po.capacity(1000) == 32 * ((1000 + 1024 + 31) // 32)
    assert po.capacity(1000000) == 32 * ((1000000 + 8000 + 31) // 32)
    assert o.capacity == po.capacity(64)


# ---------------------------------------------------------------------------------------------
# O10 adaptive step  <-  Eq. 8 (L115-L118)
# ---------------------------------------------------------------------------------------------

def test_overlap_closed_form_range_and_monotonicity():
    rng = np.random.default_rng(6)
    N = 4096
    E = (-2 * N + 4 * rng.integers(500, 900, 2000)).astype(np.int32)
    assert po.overlap_of(2000, E, 0.0) == 1.0                        # w = 1: alpha = min(1, R/R_cur)
    assert po.overlap_of(1500, E, 0.0) == pytest.approx(0.75, rel=1e-15)
    assert po.overlap_of(3000, E, 0.0) == 1.0
    grid = np.linspace(0, 0.05, 60)
    a = np.array([po.overlap_of(2000, E, d) for d in grid])
    assert np.all(a >= 0) and np.all(a <= 1 + 1e-15)                 # L118
    assert np.all(np.diff(a) <= 1e-12)
    # Eq. 8 written out directly in high precision
    import mpmath as mp
    d = 0.01
    Q = mp.fsum(mp.exp(-mp.mpf(d) * int(e)) for e in E) / 2000
    alpha = mp.fsum(min(mp.mpf(1), 2000 * mp.exp(-mp.mpf(d) * int(e)) / (2000 * Q)) for e in E) / 2000
    assert po.overlap_of(2000, E, d) == pytest.approx(float(alpha), rel=1e-12)


def test_adapt_dbeta_brackets_the_target():
    L, R = 8, 3000
    o = po.Oracle(L, R, 8)
    o.sweep(0.2, 5)
    target = 0.85
    d = o.adapt_dbeta(target, 0.2, 1.0)
    hi = 1.0 - 0.2
    assert 0 < d < hi
    assert o.overlap(d) >= target
    assert o.overlap(d + hi * 2.0**-39) < target
    # state untouched
    assert o.population == R and o.resample_counter == 0
    # a target the whole interval satisfies returns the interval
    o2 = po.Oracle(L, R, 8)
    assert o2.adapt_dbeta(0.5, 0.0, 1e-6) == 1e-6
    # EXACTLY 40 halvings of [0, hi], the lower end returned (O10): with hi = 1 every midpoint is a dyadic fraction, so the result is
    # an integer multiple of 2^-40 and the bracket's upper end, one unit above, fails the target.  39 steps would leave the upper end
    # passing on about half of the populations, 41 steps a non-integer multiple on about half: six populations
    for seed in range(9, 15):
        o3 = po.Oracle(L, R, seed)
        d3 = o3.adapt_dbeta(target, 0.0, 1.0)
        k = d3 * 2.0**40
        assert 0 < d3 < 1 and k == math.floor(k), seed
        assert o3.overlap(d3) >= target > o3.overlap(d3 + 2.0**-40), seed


# ---------------------------------------------------------------------------------------------
# whole method (O3 + O5-O8)  <-  exact results: L = 4 enumeration, Kaufman at L = 16
# ---------------------------------------------------------------------------------------------

def _seed_scatter(L, R, betas, theta, seeds, hist=False):
    runs, pops = [], []
    for s in seeds:
        o = po.Oracle(L, R, s)
        runs.append(pa_driver.run_fixed(o, betas, theta, hist=hist))
        pops.append(o)
    return runs, pops


def test_pa_run_matches_exact_enumeration_L4():
    L, R, theta = 4, 4000, 5
    betas = [i / 40 for i in range(41)]                               # 0 .. 1
    seeds = list(range(100, 116))                                    # north_star: 4 sigma; >= 16 seeds
    runs, pops = _seed_scatter(L, R, betas, theta, seeds, hist=True)
    for i in (4, 12, 18, 24, 40):
        exact = ex.exact_small(betas[i], L)
        for key in ("e", "C", "absm", "m2", "m4", "betaF_per_N", "S_per_N"):
            vals = np.array([r[i][key] for r in runs])
            sigma = vals.std(ddof=1) / math.sqrt(len(seeds))
            assert abs(vals.mean() - exact[key]) < 4 * sigma + 1e-12, (betas[i], key, vals.mean(), exact[key], sigma)
    # population size stays close to R (L69): every r_j is a Bernoulli rounding
    for r in runs:
        assert all(abs(o["R"] - R) <= 4 * math.sqrt(R) / 2 * 1.5 for o in r)
    # O9 multi-histogram (Eq. 9): ln Omega(E) against the exact density of states
    g = ex.density_of_states(L)
    N = L * L
    errs = []
    for o in pops:
        H, lnD = o.histogram()
        assert H.sum() == sum(x["R"] for x in runs[pops.index(o)])   # sum_E P(E) = R_i at every beta (L127)
        for m in range(N + 1):
            Em = -2 * N + 4 * m
            if Em not in g:
                assert H[m] == 0                                      # E = +-28 do not exist on the 4x4 torus
            elif Em <= 12:                                            # levels every run visits often
                assert H[m] > 50
                errs.append((math.log(H[m]) - lnD[m]) - math.log(g[Em]))
    errs = np.array(errs).reshape(len(pops), -1)
    sig = errs.std(0, ddof=1) / math.sqrt(len(pops))
    assert np.all(np.abs(errs.mean(0)) < 4 * sig + 5e-3), (errs.mean(0), sig)
    assert np.abs(errs.mean(0)).max() < 0.05


def test_pa_run_matches_kaufman_L16(cfg1_oracle_runs):
    # configs[0] of BASELINE.json (L=16, R=1000, 100 steps, theta=10) over 16 seeds, 4 sigma (runs shared with other pins: conftest.py)
    L = 16
    betas, shared = cfg1_oracle_runs
    runs = [obs for _, obs in shared]
    seeds = list(range(len(runs)))
    for i in (10, 30, 44, 60, 100):
        k = ex.kaufman(betas[i], L)
        for key in ("e", "C", "betaF_per_N", "S_per_N"):
            vals = np.array([r[i][key] for r in runs])
            sigma = vals.std(ddof=1) / math.sqrt(len(seeds))
            assert abs(vals.mean() - k[key]) < 4 * sigma + 1e-9, (betas[i], key, vals.mean(), k[key], sigma)
        # Eq. 4 (L90): sum_k ln Q_k estimates ln Z(beta) - N ln 2
        lnZ_est = np.array([-r[i]["betaF_per_N"] * L * L for r in runs])
        assert abs(lnZ_est.mean() - k["lnZ"]) < 4 * lnZ_est.std(ddof=1) / math.sqrt(len(seeds))
        # magnetisation symmetry is not broken by the dynamics: <|m|> in [0,1], m2 >= absm^2
        for r in runs:
            assert 0 <= r[i]["absm"] <= 1 and r[i]["m2"] >= r[i]["absm"] ** 2 - 1e-12


def test_observables_definitions_on_a_known_population():
    # Eq. 3 (L77-L86) on a population whose E_j, M_j are known in closed form
    L, N, R = 4, 16, 6
    o = po.Oracle(L, R, 1)
    yy, xx = np.divmod(np.arange(N), L)
    up = np.ones(N, dtype=np.int8)
    cb = (((xx + yy) & 1) * 2 - 1).astype(np.int8)
    one = up.copy(); one[5] = -1                                       # one flipped spin: E = -2N+8, M = N-2
    o.set_spins(0, np.stack([up, -up, cb, one, -one, up]))
    E, M = o.energies()
    assert E.tolist() == [-32, -32, 32, -24, -24, -32] and M.tolist() == [16, -16, 0, 14, -14, 16]
    beta = 0.37
    obs = o.observables(beta)
    Ef = np.array(E, dtype=np.float64); Mf = np.array(M, dtype=np.float64)
    assert obs["e"] == pytest.approx(Ef.mean() / N, rel=1e-15)
    assert obs["C"] == pytest.approx(beta**2 * N * ((Ef / N) ** 2).mean() - beta**2 * N * (Ef.mean() / N) ** 2, rel=1e-12)
    assert obs["absm"] == pytest.approx(np.abs(Mf).mean() / N, rel=1e-15)
    assert obs["m2"] == pytest.approx(((Mf / N) ** 2).mean(), rel=1e-15)
    assert obs["m4"] == pytest.approx(((Mf / N) ** 4).mean(), rel=1e-15)
    assert obs["S_per_N"] == pytest.approx(beta * obs["e"] - obs["betaF_per_N"], rel=1e-15)   # Eq. 5


def test_histogram_invariants():
    L, R = 8, 2000
    N = L * L
    o = po.Oracle(L, R, 21)
    betas = [0.0, 0.1, 0.2, 0.3]
    tot = 0
    SE_tot = 0
    o.hist_accumulate(0.0); tot += o.population; SE_tot += int(o.energies()[0].astype(np.int64).sum())
    for i in range(1, 4):
        o.resample(betas[i - 1], betas[i]); o.sweep(betas[i], 3); o.hist_accumulate(betas[i])
        tot += o.population
        SE_tot += int(o.energies()[0].astype(np.int64).sum())
    H, lnD = o.histogram()
    assert H.sum() == tot                                              # L127
    Em = -2 * N + 4 * np.arange(N + 1)
    assert int((H * Em).sum()) == SE_tot
    assert np.all(np.isfinite(lnD))
    # first denominator term alone: R_0 * exp(-N ln 2 - 0) at beta_0 = 0
    o2 = po.Oracle(L, R, 21); o2.hist_accumulate(0.0)
    assert np.allclose(o2.histogram()[1], math.log(R) - N * math.log(2), rtol=1e-15)


def test_determinism_same_seed_same_bytes():
    # "provably simulates the same set of configurations in each run"
    outs = []
    for _ in range(2):
        o = po.Oracle(8, 500, 42)
        obs = pa_driver.run_fixed(o, [0.0, 0.1, 0.2, 0.3], 4)
        outs.append((o.get_spins().tobytes(), repr(obs)))
    assert outs[0] == outs[1]
