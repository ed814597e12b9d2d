"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs (-m gpu).  Bar: bit-exact for spins, energies, copy numbers, offsets, R_new and
histogram counts; relative 1e-9 for fp64 observables (BASELINE.json north_star)."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("no CUDA device", allow_module_level=True)

from oracle import pa_oracle as po                      # noqa: E402
from paper_1703_03676_b200 import pa                    # noqa: E402
from paper_1703_03676_b200.workloads import CONFIGS     # noqa: E402
import pa_driver                                        # noqa: E402

REL = 1e-9
OBS_KEYS = ("beta", "e", "C", "absm", "m2", "m4", "betaF_per_N", "S_per_N", "lnQ")


def assert_obs_close(a, b):
    assert a["R"] == b["R"]
    for k in OBS_KEYS:
        assert a[k] == pytest.approx(b[k], rel=REL, abs=1e-300), (k, a[k], b[k])


def assert_same_state(g, o, full=True):
    assert g.population == o.population
    assert g.sweep_counter == o.sweep_counter and g.resample_counter == o.resample_counter
    if full:
        assert np.array_equal(g.get_spins(), o.get_spins())
    Eg, Mg = g.energies()
    Eo, Mo = o.energies()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)


# ---------------------------------------------------------------------------------------------
# a0 init, ragged populations
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("L,R,seed", [(4, 1, 3), (4, 33, 4), (6, 100, 5), (16, 1000, 1), (64, 257, 2**40 + 7)])
def test_init_bit_exact(L, R, seed):
    g, o = pa.Population(L, R, seed), po.Oracle(L, R, seed)
    assert g.capacity == o.capacity
    assert_same_state(g, o)
    assert g.lnZ == o.lnZ
    # interchange layout: word (g, s) bit b = replica 32g+b at site s
    words = g.get_words()
    sp = o.get_spins()
    j = R - 1
    bits = (words[j >> 5] >> np.uint32(j & 31)) & 1
    assert np.array_equal(bits.astype(np.int8) * 2 - 1, sp[j])
    if R % 32:
        assert np.all(words[-1] >> np.uint32(R % 32) == 0)          # unused lanes are zero


# ---------------------------------------------------------------------------------------------
# a2 sweep: per call, several tile geometries (one CTA per group, clusters of 2/4 with DSMEM halos)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("L,R", [(4, 40), (6, 70), (10, 33), (16, 200), (32, 100), (64, 96), (128, 64), (256, 40), (192, 40), (512, 33)])
def test_sweep_bit_exact(L, R):
    seed = 1000 + L
    g, o = pa.Population(L, R, seed), po.Oracle(L, R, seed)
    for beta, theta in [(0.0, 1), (0.3, 2), (0.4406868, 3), (1.0, 1), (0.7, 0)]:
        g.sweep(beta, theta); o.sweep(beta, theta)
        assert_same_state(g, o)


@pytest.mark.parametrize("L,R", [(4, 40), (6, 70), (10, 33), (16, 200), (32, 100), (64, 96), (128, 64), (256, 40), (192, 40), (512, 33)])
def test_sweep_lcg_mode_bit_exact(L, R):
    """LCG-assisted stream (O11): generic kernel (L < 64 or not a power of two) and the
    quad-row column-walk kernel, ragged last group, switching modes between calls."""
    seed = 2000 + L
    g, o = pa.Population(L, R, seed), po.Oracle(L, R, seed)
    g.set_rng_mode(pa.PA_RNG_LCG); o.set_rng_mode(po.RNG_LCG)
    assert g.rng_mode == pa.PA_RNG_LCG
    for beta, theta in [(0.0, 1), (0.3, 2), (0.4406868, 3), (1.0, 1), (0.7, 0)]:
        g.sweep(beta, theta); o.sweep(beta, theta)
        assert_same_state(g, o)
    g.set_rng_mode(pa.PA_RNG_PHILOX); o.set_rng_mode(po.RNG_PHILOX)
    g.sweep(0.5, 1); o.sweep(0.5, 1)
    assert_same_state(g, o)
    rc = pa.lib().pa_set_rng_mode(g._h, 2)
    assert rc == pa.PA_ERR_INVALID_ARG and g.rng_mode == pa.PA_RNG_PHILOX


def test_sweep_lcg_mode_geometries(monkeypatch):
    """Same bytes for every launch geometry (clusters of 1/2/4/8 CTAs with DSMEM halos, 128/256 threads), all
    equal to the oracle."""
    L, R, seed = 64, 130, 77
    o = po.Oracle(L, R, seed); o.set_rng_mode(po.RNG_LCG)
    o.sweep(0.42, 3)
    want = o.get_spins()
    for env in ({}, {"PA_SWEEP_C": "2"}, {"PA_SWEEP_C": "4", "PA_SWEEP_T": "128"}, {"PA_SWEEP_C": "8", "PA_SWEEP_T": "64"},
                {"PA_SWEEP_C": "4"}, {"PA_SWEEP_KIND": "0"}, {"PA_SWEEP_KIND": "0", "PA_SWEEP_C": "2", "PA_SWEEP_T": "96"}):
        for k in ("PA_SWEEP_C", "PA_SWEEP_T", "PA_SWEEP_KIND"):
            monkeypatch.delenv(k, raising=False)
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        g = pa.Population(L, R, seed); g.set_rng_mode(pa.PA_RNG_LCG)
        g.sweep(0.42, 3)
        assert np.array_equal(g.get_spins(), want), env


def test_lcg_mode_whole_run_config1():
    """configs[0] (L=16, R=1000, 100 steps, theta=10) with the LCG-assisted sweeps: every step bit-exact."""
    wl = CONFIGS[1]
    g, o = pa.Population(wl.L, wl.R, wl.seed), po.Oracle(wl.L, wl.R, wl.seed)
    g.set_rng_mode(pa.PA_RNG_LCG); o.set_rng_mode(po.RNG_LCG)
    betas = wl.betas()
    og = pa_driver.run_fixed(g, betas, wl.theta, on_step=lambda i, p: None)
    oo = pa_driver.run_fixed(o, betas, wl.theta)
    for a, b in zip(og, oo):
        assert_obs_close(a, b)
    assert_same_state(g, o)


def test_sweep_split_calls_and_special_states():
    L, R = 16, 64
    g, o = pa.Population(L, R, 9), po.Oracle(L, R, 9)
    N = L * L
    yy, xx = np.divmod(np.arange(N), L)
    states = np.stack([np.ones(N), -np.ones(N), ((xx + yy) & 1) * 2 - 1, (yy & 1) * 2 - 1]).astype(np.int8)
    g.set_spins(3, states); o.set_spins(3, states)
    assert_same_state(g, o)
    E, M = g.energies()
    assert E[3:7].tolist() == [-2 * N, -2 * N, 2 * N, 0] and M[3:7].tolist() == [N, -N, 0, 0]
    # theta = 5 in one call on the GPU, 2 + 3 on the oracle: the sweep counter carries the stream
    g.sweep(0.5, 5)
    o.sweep(0.5, 2); o.sweep(0.5, 3)
    assert_same_state(g, o)


# ---------------------------------------------------------------------------------------------
# a4-a7 resample chain, per step
# ---------------------------------------------------------------------------------------------

def _compare_resample(g, o, beta, beta_new):
    R_prev = g.population
    Rg = g.resample(beta, beta_new)
    Ro = o.resample(beta, beta_new)
    assert Rg == Ro
    dg, do = g.resample_debug(R_prev), o.resample_debug(R_prev)
    assert dg["W"] == do["W"]                                        # fixed-order fp64 sum: bit-exact
    assert np.array_equal(dg["w"], do["w"])
    assert np.array_equal(dg["r"], do["r"])
    assert np.array_equal(dg["o"], do["o"])
    assert g.lnZ == pytest.approx(o.lnZ, rel=1e-15)


@pytest.mark.parametrize("L,R", [(8, 50), (16, 1000), (16, 3333), (64, 2500)])
def test_resample_chain_bit_exact(L, R):
    g, o = pa.Population(L, R, 31), po.Oracle(L, R, 31)
    beta = 0.0
    for step, db in enumerate([0.0, 0.05, 0.1, 0.02, 0.3]):
        _compare_resample(g, o, beta, beta + db)
        beta += db
        assert_same_state(g, o)
        g.sweep(beta, 2); o.sweep(beta, 2)
        assert_same_state(g, o)
        assert_obs_close(g.observables(beta), o.observables(beta))


@pytest.mark.parametrize("L,R", [(16, 4133), (8, 700), (64, 777)])
def test_copy_strong_resampling(L, R):
    """Copy kernel under strong resampling: many empty and many-fold copy numbers, parents spanning several
    source groups, ragged last group; N/4 below, at and above two chunks per thread."""
    g, o = pa.Population(L, R, 9), po.Oracle(L, R, 9)
    beta = 0.0
    for db in (0.03, 0.25, 0.4, 0.0, 1.5):
        _compare_resample(g, o, beta, beta + db)
        beta += db
        assert_same_state(g, o)
        g.sweep(beta, 1); o.sweep(beta, 1)


@pytest.mark.parametrize("L,R", [(4, 1), (4, 2), (6, 32), (8, 33), (4, 5000)])
def test_tiny_and_ragged_populations_whole_run(L, R):
    """Degenerate population sizes: a single replica (r_0 is always 1 because tau = R w / W = 1), exactly one word, one word
    plus one replica, and a lattice of 4 chunks (fewer 128-bit chunks than copy threads)."""
    g, o = pa.Population(L, R, 17), po.Oracle(L, R, 17)
    betas = [0.0, 0.2, 0.45, 0.9]
    og = pa_driver.run_fixed(g, betas, 3, hist=True)
    oo = pa_driver.run_fixed(o, betas, 3, hist=True)
    for a, b in zip(og, oo):
        assert_obs_close(a, b)
    assert_same_state(g, o)
    assert np.array_equal(g.histogram()[0], o.histogram()[0])
    d_g, d_o = g.adapt_dbeta(0.7, 0.9, 2.0), o.adapt_dbeta(0.7, 0.9, 2.0)
    assert d_g == d_o


def test_resample_identity_capacity_and_errors():
    L, R = 16, 500
    g, o = pa.Population(L, R, 5), po.Oracle(L, R, 5)
    before = g.get_spins()
    assert g.resample(0.0, 0.0) == R                                 # dbeta = 0: r = 1, identity copy
    assert np.array_equal(g.get_spins(), before)
    rc, _ = g.resample_rc(0.5, 0.4)
    assert rc == pa.PA_ERR_INVALID_ARG
    # shrink the population to a handful of replicas, then resample: R_new ~ R_target >> R_cur
    g.sweep(0.3, 3); o.sweep(0.3, 3)
    words = g.get_words()
    g.set_words(70, words[:3])
    sp = g.get_spins()
    # the oracle has no set_words: compare with the plan computed from the energies instead
    E, _ = g.energies()
    plan = po.resample_plan(R, E, 5, g.resample_counter, 0.31 - 0.3)
    R_prev = g.population
    assert g.resample(0.3, 0.31) == plan["R_new"]
    d = g.resample_debug(R_prev)
    assert np.array_equal(d["r"], plan["r"]) and np.array_equal(d["o"], plan["o"]) and d["W"] == plan["W"]
    parent = np.repeat(np.arange(R_prev), plan["r"])
    assert np.array_equal(g.get_spins(), sp[parent])


# ---------------------------------------------------------------------------------------------
# whole runs
# ---------------------------------------------------------------------------------------------

def test_config1_full_run_every_step():
    """BASELINE.json configs[0]: L=16, R=1000, beta 0..1 in 100 steps, theta=10, seed 1."""
    wl = CONFIGS[1]
    g, o = pa.Population(wl.L, wl.R, wl.seed), po.Oracle(wl.L, wl.R, wl.seed)
    betas = wl.betas()
    assert_obs_close(g.observables(betas[0]), o.observables(betas[0]))
    for i in range(1, len(betas)):
        _compare_resample(g, o, betas[i - 1], betas[i])
        g.sweep(betas[i], wl.theta); o.sweep(betas[i], wl.theta)
        assert_same_state(g, o)
        assert_obs_close(g.observables(betas[i]), o.observables(betas[i]))


def test_config2_first_steps():
    """BASELINE.json configs[1]: L=64, R=20000, dbeta=0.005, theta=10, seed 2 (first 3 steps in full)."""
    wl = CONFIGS[2]
    g, o = pa.Population(wl.L, wl.R, wl.seed), po.Oracle(wl.L, wl.R, wl.seed)
    betas = wl.betas()
    for i in range(1, 4):
        _compare_resample(g, o, betas[i - 1], betas[i])
        g.sweep(betas[i], wl.theta); o.sweep(betas[i], wl.theta)
        assert_same_state(g, o)
        assert_obs_close(g.observables(betas[i]), o.observables(betas[i]))


def test_adaptive_run_with_multihistogram():
    """The adaptive schedule and Eq. 9 accumulation (shape of configs[3], scaled to L=16, R=2000)."""
    L, R, seed, theta, target = 16, 2000, 4, 3, 0.85
    g, o = pa.Population(L, R, seed), po.Oracle(L, R, seed)
    bg, og = pa_driver.run_adaptive(g, 0.0, 0.6, theta, target, hist=True, max_steps=25)
    bo, oo = pa_driver.run_adaptive(o, 0.0, 0.6, theta, target, hist=True, max_steps=25)
    assert bg == bo                                                  # the beta sequence is bit-identical
    assert len(bg) > 5
    for a, b in zip(og, oo):
        assert_obs_close(a, b)
    assert_same_state(g, o)
    Hg, Dg = g.histogram()
    Ho, Do = o.histogram()
    assert np.array_equal(Hg, Ho)
    fin = np.isfinite(Do)
    assert np.array_equal(np.isfinite(Dg), fin)
    assert np.allclose(Dg[fin], Do[fin], rtol=REL, atol=0)
    # the overlap function itself
    for d in (0.0, 0.003, 0.02):
        assert g.overlap(d) == o.overlap(d)
    # O12: reweighting of the accumulated sums to a fine beta grid (Sec. 2.4), inside and beyond the simulated range
    grid = np.concatenate([np.linspace(0.0, bg[-1], 37), [bg[-1] + 0.05, 1.5]])
    rg, ro = g.reweight(grid), {**o.reweight(grid), **o.reweight_mag(grid)}
    for k in ("lnZ", "e", "C", "absm", "m2"):
        assert np.allclose(rg[k], ro[k], rtol=REL, atol=1e-300), k
    # O14: the microcanonical magnetisation sums are exact integers
    for a, b in zip(g.mag_sums(), o.mag_sums()):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("L,R,seed,coupl", [(16, 2000, 4, False), (32, 50000, 5, False), (8, 3, 6, False), (64, 20000, 7, False),
                                             (16, 5000, 8, True), (128, 4000, 9, False)])
def test_adaptive_filter_equals_exact_path(monkeypatch, L, R, seed, coupl):
    """O10: pa_adapt_dbeta takes most of its 41 decisions on the energy histogram inside one kernel and hands only those within
    the rounding bound of the target to the exact evaluation (csrc/pa_adapt.cu).  Its result must equal, bit for bit, the
    41 exact evaluations (PA_ADAPT_EXACT=1) and the oracle's, for every target, bracket and temperature tried -- including
    brackets whose upper end already satisfies the target and targets the population cannot reach."""
    from paper_1703_03676_b200.workloads import random_couplings
    g, o = pa.Population(L, R, seed), po.Oracle(L, R, seed)
    if coupl:
        Jx, Jy = random_couplings(L, seed)
        g.set_couplings(Jx, Jy); o.set_couplings(Jx, Jy)
    beta = 0.0
    total_exact = total_calls = 0
    for step in range(6):
        E, _ = g.energies()
        for target, bmax in ((0.85, beta + 1.0), (0.5, beta + 1.0), (0.97, beta + 0.3), (0.3, beta + 1e-4), (0.999999, beta + 2.0), (0.05, beta + 40.0)):
            g.set_switch("PA_ADAPT_EXACT", None)                       # (the environment is read at pa_create only)
            d_f = g.adapt_dbeta(target, beta, bmax)
            n_exact, n_launch = g.adapt_stats()
            margin, _ = g.adapt_margins()
            assert margin > 1.0                                        # a decision of the filter is never inside its threshold
            g.set_switch("PA_ADAPT_EXACT", 1)
            d_e = g.adapt_dbeta(target, beta, bmax)
            assert g.adapt_stats()[0] in (1, 41)
            d_o = po.adapt_dbeta_of(R, E, target, beta, bmax)
            assert d_f == d_e == d_o, (step, target, bmax, d_f, d_e, d_o)
            assert n_launch >= 1 and n_exact <= 12, (n_exact, n_launch)
            total_exact += n_exact; total_calls += 1
        g.set_switch("PA_ADAPT_EXACT", None)
        d = g.adapt_dbeta(0.85, beta, beta + 1.0)
        assert d == o.adapt_dbeta(0.85, beta, beta + 1.0)
        g.resample(beta, beta + d); o.resample(beta, beta + d)
        beta += d
        g.sweep(beta, 2); o.sweep(beta, 2)
    assert total_exact < 6 * total_calls                              # a handful per call instead of 41
    assert g.adapt_margins()[1] < 4.0                                 # |alpha' - alpha| at every hand-back, in first-order bounds (threshold: 4)
    assert_same_state(g, o)


def test_reweight_errors_and_device_buffers():
    L, R = 8, 300
    g, o = pa.Population(L, R, 3), po.Oracle(L, R, 3)
    grid = np.array([0.1, 0.2])
    rc = pa.lib().pa_reweight(g._h, 2, pa._ptr(grid), None, None, None, None, None)
    assert rc == pa.PA_ERR_INVALID_ARG                                # nothing accumulated yet
    obs_g = pa_driver.run_fixed(g, [0.0, 0.1, 0.2, 0.3], 2, hist=True)
    pa_driver.run_fixed(o, [0.0, 0.1, 0.2, 0.3], 2, hist=True)
    assert pa.lib().pa_reweight(g._h, 0, pa._ptr(grid), None, None, None, None, None) == pa.PA_ERR_INVALID_ARG
    want = o.reweight(grid)
    tb = torch.tensor(grid, device="cuda"); te = torch.empty(2, dtype=torch.float64, device="cuda")
    assert pa.lib().pa_reweight(g._h, 2, pa._ptr(tb), None, pa._ptr(te), None, None, None) == pa.PA_OK
    torch.cuda.synchronize()
    assert np.allclose(te.cpu().numpy(), want["e"], rtol=REL)
    assert g.population == obs_g[-1]["R"]                             # state untouched


def test_weighted_average_of_runs():
    """O13 (Eq. 6-7): M independent GPU populations combined by their free-energy estimates."""
    L, R, M = 8, 200, 6
    betas = [0.0, 0.15, 0.3, 0.45]
    lnZ, A = [], []
    for m in range(M):
        g = pa.Population(L, R, 900 + m)
        ob = pa_driver.run_fixed(g, betas, 2)[-1]
        lnZ.append(g.lnZ); A.append([ob["e"], ob["C"], ob["absm"]])
    out_g, w_g = pa.pa_weighted_average(lnZ, A)
    out_o, w_o = po.weighted_average(lnZ, A)
    assert np.allclose(w_g, w_o, rtol=REL) and np.allclose(out_g, out_o, rtol=REL)
    assert abs(w_g.sum() - 1) < 1e-12
    big = np.array([800.0, 0.0, -800.0])
    out_g, w_g = pa.pa_weighted_average(big, np.arange(3.0)[:, None])
    assert w_g.tolist() == [1.0, 0.0, 0.0] and out_g[0] == 0.0


def test_adaptive_multi_run_protocol_first_run_decides():
    """PAPER.md L118 (Sec. 2.3) + Eq. 6-7 (L99-L109): in adaptive mode the first run decides the temperature steps and the remaining
    runs keep its sequence, so that the runs can be averaged at every temperature.  Run A anneals adaptively and records its
    betas; runs B and C (other seeds) follow A's list -- B through the single calls, C through one pa_anneal call; the
    free-energy-weighted averages of (A, B, C) at three of A's temperatures equal the oracle's on its own three runs."""
    L, R, theta, target = 16, 600, 3, 0.8
    seeds = (1201, 1202, 1203)

    def three_runs(make, anneal_third):
        a = make(seeds[0])
        betas, obs_a = pa_driver.run_adaptive(a, 0.0, 0.6, theta, target)
        lnz_a = []
        a2 = make(seeds[0])                                            # lnZ of run A at every temperature: replay A on its own list
        pa_driver.run_fixed(a2, betas, theta, on_step=lambda i, p: lnz_a.append(p.lnZ))
        assert a2.lnZ == a.lnZ
        lnz_b, b = [], make(seeds[1])
        obs_b = pa_driver.run_fixed(b, betas, theta, on_step=lambda i, p: lnz_b.append(p.lnZ))
        c = make(seeds[2])
        if anneal_third:
            obs_c = [c.observables(betas[0])] + c.anneal(betas, theta)
        else:
            obs_c = pa_driver.run_fixed(c, betas, theta)
        lnz_c = [-obs_c[i]["betaF_per_N"] * L * L for i in range(1, len(betas))]          # ln Z = -beta F (Eq. 4)
        return betas, (obs_a, obs_b, obs_c), (lnz_a, lnz_b, lnz_c)

    bg, og, zg = three_runs(lambda s: pa.Population(L, R, s), True)
    bo, oo, zo = three_runs(lambda s: po.Oracle(L, R, s), False)
    assert bg == bo and len(bg) >= 6                                    # the schedule itself is bit-exact (O10)
    for i in (1, len(bg) // 2, len(bg) - 1):
        keys = ("e", "C", "absm", "m2", "m4")
        Ag = [[o[i][k] for k in keys] for o in og]
        Ao = [[o[i][k] for k in keys] for o in oo]
        lg = [z[i - 1] for z in zg]
        lo = [z[i - 1] for z in zo]
        assert np.allclose(lg, lo, rtol=REL)
        out_g, w_g = pa.pa_weighted_average(lg, Ag)
        out_o, w_o = po.weighted_average(lo, Ao)
        assert np.allclose(w_g, w_o, rtol=REL) and np.allclose(out_g, out_o, rtol=REL)
        assert 0 < w_g.min() and abs(w_g.sum() - 1) < 1e-12


def test_handles_on_two_devices_need_no_set_device():
    """A handle belongs to the device it was created on and every call makes that device current for its own duration
    (include/pa.h, pa_create): two populations on two GPUs driven from one thread without switching devices in between, the
    caller's current device untouched, results equal to the oracle's."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    pops = []
    for dev in (0, 1):
        with torch.cuda.device(dev):
            pops.append(pa.Population(16, 500, 70 + dev, own_memory=True))
    torch.cuda.set_device(0)
    betas = [0.0, 0.2, 0.4]
    for dev, g in enumerate(pops):                                     # device 0 stays current throughout
        o = po.Oracle(16, 500, 70 + dev)
        og, oo = pa_driver.run_fixed(g, betas, 2), pa_driver.run_fixed(o, betas, 2)
        assert torch.cuda.current_device() == 0
        assert_same_state(g, o)
        assert_obs_close(og[-1], oo[-1])
    lnZ = [g.lnZ for g in pops]
    out, w = pa.pa_weighted_average(lnZ, [[g.observables(betas[-1])["e"]] for g in pops])      # Eq. 6-7 over GPUs
    assert abs(w.sum() - 1) < 1e-12


def test_switches_are_read_at_create_only(monkeypatch):
    """The environment is read once, in pa_create*: changing it afterwards does not reach a live handle (pa_set_switch does)."""
    monkeypatch.delenv("PA_SWEEP_KIND", raising=False)
    g = pa.Population(64, 64, 5)
    monkeypatch.setenv("PA_SWEEP_KIND", "0")
    g.sweep(0.3, 1)
    assert g.last_sweep_kind & pa.PA_SWEEP_RAN_COL                     # still the column-walk kernel
    g2 = pa.Population(64, 64, 5)
    g2.sweep(0.3, 1)
    assert not g2.last_sweep_kind & pa.PA_SWEEP_RAN_COL                # a handle created under the variable took it
    g.set_switch("PA_SWEEP_KIND", 0)
    g3 = pa.Population(64, 64, 5)
    g3.set_switch("PA_SWEEP_KIND", None)
    g.sweep(0.3, 1); g2.sweep(0.3, 1); g3.sweep(0.3, 2)
    assert not g.last_sweep_kind & pa.PA_SWEEP_RAN_COL and g3.last_sweep_kind & pa.PA_SWEEP_RAN_COL
    assert np.array_equal(g.get_spins(), g2.get_spins()) and np.array_equal(g.get_spins(), g3.get_spins())
    with pytest.raises(pa.PaError):
        g.set_switch("PA_NO_SUCH_SWITCH", 1)


def test_determinism_and_geometry_independence(monkeypatch):
    """Same seed -> same bytes; a different launch geometry -> same bytes."""
    outs = []
    for env in ({}, {}, {"PA_SWEEP_C": "2", "PA_SWEEP_T": "64"}, {"PA_SWEEP_C": "4", "PA_SWEEP_T": "128", "PA_SWEEP_CMP": "0"}):
        for k in ("PA_SWEEP_C", "PA_SWEEP_T", "PA_SWEEP_CMP"):
            monkeypatch.delenv(k, raising=False)
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        g = pa.Population(32, 300, 77)
        obs = pa_driver.run_fixed(g, [0.0, 0.2, 0.4, 0.5], 3)
        outs.append((g.get_spins().tobytes(), repr(obs)))
    assert outs[0] == outs[1] == outs[2] == outs[3]


def test_sweep_threshold_extremes():
    """T = 2^32-1 (beta = 0), tiny thresholds and T8 = 0 (beta = 3: exp(-24) 2^32 < 1) on both compare paths."""
    L, R = 8, 96
    for beta in (0.0, 3.0, 5.0, 2.7):
        g, o = pa.Population(L, R, 123), po.Oracle(L, R, 123)
        assert po.thresholds(3.0)[1] == 0
        g.sweep(0.2, 1); o.sweep(0.2, 1)
        g.sweep(beta, 3); o.sweep(beta, 3)
        assert_same_state(g, o)


@pytest.mark.parametrize("L,R,mode,coupl", [(16, 1000, 0, False), (6, 70, 0, False), (10, 161, 0, True), (32, 100, 0, False), (4, 33, 0, False),
                                             (16, 1000, 1, False), (12, 161, 1, True), (32, 100, 1, False), (8, 70, 1, False)])
def test_sweep_lane_split_kernel(monkeypatch, L, R, mode, coupl):
    """Small populations on the generic path: S = 2, 4 lane-split CTAs per group, each running 8/S of every word's Philox calls
    (or, in the LCG-assisted stream, jumping to the outputs of its lanes) and writing back only its own bytes of the words -- the
    same bytes as one CTA per group and as the oracle (thresholds at beta = 0 and at a T8 of 0 included; R = 1000 at L = 16 is
    configs[0]'s population, R = 161 has a ragged last word; ferromagnet and random +-J couplings)."""
    from paper_1703_03676_b200.workloads import random_couplings
    seed = 4000 + L
    o = po.Oracle(L, R, seed)
    o.set_rng_mode(mode)
    if coupl:
        Jx, Jy = random_couplings(L, seed)
        o.set_couplings(Jx, Jy)
    plan = [(0.0, 1), (0.3, 2), (0.4406868, 3), (3.0, 1), (0.7, 2)]
    for beta, theta in plan:
        o.sweep(beta, theta)
    want, (Eo, Mo) = o.get_spins(), o.energies()
    for split in ("0", "2", "4", None):
        monkeypatch.delenv("PA_SWEEP_SPLIT", raising=False)
        if split is not None:
            monkeypatch.setenv("PA_SWEEP_SPLIT", split)
        g = pa.Population(L, R, seed)
        g.set_rng_mode(mode)
        if coupl:
            g.set_couplings(Jx, Jy)
        for beta, theta in plan:
            g.sweep(beta, theta)
        assert np.array_equal(g.get_spins(), want), split
        Eg, Mg = g.energies()
        assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo), split
        words = g.get_words()
        if R % 32:
            assert np.all(words[-1] >> np.uint32(R % 32) == 0)


@pytest.mark.parametrize("L,R,rng", [(64, 5300, 0), (64, 5300, 1), (64, 9500, 0), (128, 4800, 0), (128, 4800, 1)])
def test_sweep_mixed_launch(monkeypatch, L, R, rng):
    """Medium populations on the column-walk kernels: whole groups (one per CTA) fill complete rounds of the 148 SMs and the
    remaining groups are split over the CTAs of a cluster -- one launch, the same bytes as the uniform launch and the oracle.
    Sampled slots span the whole groups, the first and last split group and the ragged last word."""
    seed = 5000 + L + rng
    o = po.Oracle(L, R, seed)
    o.set_rng_mode(po.RNG_LCG if rng else po.RNG_PHILOX)
    o.sweep(0.35, 1); o.sweep(0.45, 2)
    want = o.get_spins()
    Eo, Mo = o.energies()
    outs = []
    for mixed in ("1", "0"):
        monkeypatch.setenv("PA_SWEEP_MIXED", mixed)
        g = pa.Population(L, R, seed)
        g.set_rng_mode(pa.PA_RNG_LCG if rng else pa.PA_RNG_PHILOX)
        g.sweep(0.35, 1); g.sweep(0.45, 2)
        Eg, Mg = g.energies()
        assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo), mixed
        assert np.array_equal(g.get_spins(), want), mixed
        outs.append(g.get_words().tobytes())
    assert outs[0] == outs[1]


def test_words_export_import_aligned_and_unaligned_device_buffers():
    """pa_get_words / pa_set_words move a pair of sites per thread with 8-byte accesses when the caller's buffer allows it and with
    4-byte accesses otherwise: same words through a host buffer, an aligned device buffer and one that starts 4 bytes into an
    8-byte word; ragged last group (dead lanes 0); square lattice and a box."""
    for dims, R in (((64, 64), 100), ((6, 6), 70), ((6, 4, 2), 45)):
        g = pa.Population(dims[0], R, 9) if len(dims) == 2 else pa.Population.box(dims, R, 9)
        g.sweep(0.3, 2)
        host = g.get_words()
        n = host.size
        buf = torch.zeros(n + 1, dtype=torch.int32, device="cuda")
        for off in (0, 1):
            view = buf[off:off + n]
            assert (view.data_ptr() % 8 == 0) == (off == 0)
            view.zero_()
            g.get_words(view)
            assert np.array_equal(view.cpu().numpy().view(np.uint32).reshape(host.shape), host), (dims, off)
            h2 = pa.Population(dims[0], R, 10) if len(dims) == 2 else pa.Population.box(dims, R, 10)
            h2.set_words(R, view)
            assert np.array_equal(h2.get_spins(), g.get_spins()), (dims, off)
            assert np.array_equal(h2.get_words(), host)


@pytest.mark.parametrize("L,R", [(64, 130), (64, 96), (128, 70)])
def test_sweep_lcg_p64_words_opt_in(monkeypatch, L, R):
    """PA_LCG_P64=1: the LCG column-walk kernel on 64-replica words (two adjacent groups side by side; Table 1 measures
    p = 64) -- the stream is defined per 32-replica word (O11), so the bytes are the p = 32 kernel's and the
    oracle's; an odd number of groups leaves the last pair half empty."""
    seed = 6000 + L
    o = po.Oracle(L, R, seed); o.set_rng_mode(po.RNG_LCG)
    o.sweep(0.3, 2); o.sweep(0.44, 1)
    want = o.get_spins()
    for p64 in ("1", "0"):
        monkeypatch.setenv("PA_LCG_P64", p64)
        g = pa.Population(L, R, seed); g.set_rng_mode(pa.PA_RNG_LCG)
        g.sweep(0.3, 2); g.sweep(0.44, 1)
        assert np.array_equal(g.get_spins(), want), p64
