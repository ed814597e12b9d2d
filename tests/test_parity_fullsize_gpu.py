"""GPU parity at BASELINE.json's full sizes (configs 3, 4, 5), in the launch configuration bench.py times.

The oracle cannot hold these populations (cfg5: 65.5 GB of uint8 spins, ~3e6 core-seconds), so each checked
temperature step follows the chained spot-check protocol of SURVEY.md Sec. 8(c) / DESIGN.md Sec. 7:

  (i)   the FULL energy / magnetisation vectors come back from the device (4 bytes per replica); on a random
        sample of slots the oracle recomputes E_j, M_j from the exported spins (O4);
  (ii)  from the full E vector the oracle recomputes W, w_j, r_j, o_j, R_new, ln Q (O5-O7): bit-exact;
  (iii) the copy is checked on a sample of destination slots: new[d] == old[parent(d)], parent from the oracle's plan;
  (iv)  the sampled slots are swept by the oracle (same slot ids, sweep counter, thresholds) and compared bit-exactly (O3);
  (v)   observables / adaptive step / histogram fold are recomputed by the oracle from the full E, M vectors (O8-O10).

Steps that are not checked in full still have their resampling plan (W, copy numbers via R_new, ln Q) recomputed by the oracle
from the device's full E vector; every checked step starts from device state, so a divergence anywhere upstream shows as an
(i) or (iv) mismatch only if it breaks the algorithm, which is what parity means here.

The default suite runs EVERY config's whole schedule (cfg5: 500 steps, about four minutes on a B200; cfg4: the whole adaptive
run, about 400 steps); the checked-step sets are in the tests' docstrings and in DESIGN.md Sec. 7.
PA_FULLSIZE_STEPS=short stops cfg4 / cfg5 after their first steps (local runs)."""
import os

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
RUN_ALL = os.environ.get("PA_FULLSIZE_STEPS", "all") != "short"


def _sample(rng, n_total, n, always=()):
    """n distinct slots in [0, n_total): random, plus the edges (first, last, last full group boundary)."""
    fixed = [s for s in always if 0 <= s < n_total]
    pick = rng.choice(n_total, size=min(n, n_total), replace=False).tolist()
    return np.array(sorted(set(fixed + pick)), dtype=np.int64)


def _bits(spins_pm1):
    return np.ascontiguousarray((spins_pm1 > 0).astype(np.uint8))


def checked_step(g, wl, beta_prev, beta, rng, n_slots, lnZ_ref, hist=None, rng_mode=po.RNG_PHILOX):
    """One temperature step on the device with checks (i)-(v).  Returns (observables, lnZ after the step)."""
    L, N = wl.L, wl.N
    R_prev = g.population
    E, M = g.energies()
    k = g.resample_counter
    plan = po.resample_plan(wl.R, E, wl.seed, k, beta - beta_prev)                       # (ii) oracle side
    R_new = plan["R_new"]
    parent = np.repeat(np.arange(R_prev, dtype=np.int64), plan["r"])
    assert parent.size == R_new
    d = _sample(rng, R_new, n_slots, always=(0, 1, 31, 32, R_new - 1, (R_new // 32) * 32 - 1, (R_new // 32) * 32))
    pre = g.get_spins_at(parent[d])
    Eo, Mo = po.energies_of(L, _bits(pre))                                                # (i)
    assert np.array_equal(Eo, E[parent[d]]) and np.array_equal(Mo, M[parent[d]])

    assert g.resample(beta_prev, beta) == R_new                                           # (ii) device side
    dbg = g.resample_debug(R_prev)
    assert dbg["W"] == plan["W"]
    assert np.array_equal(dbg["w"], plan["w"])
    assert np.array_equal(dbg["r"], plan["r"])
    assert np.array_equal(dbg["o"], plan["o"])
    lnZ = lnZ_ref + plan["lnQ"]
    assert g.lnZ == pytest.approx(lnZ, rel=1e-13)

    post = g.get_spins_at(d)                                                              # (iii)
    assert np.array_equal(post, pre)

    t0 = g.sweep_counter                                                                  # (iv)
    g.sweep(beta, wl.theta)
    assert g.sweep_counter == t0 + wl.theta
    want = po.sweep_slots(L, wl.seed, t0, beta, wl.theta, d, _bits(post), rng_mode=rng_mode)
    got = g.get_spins_at(d)
    assert np.array_equal(_bits(got), want)

    E2, M2 = g.energies()                                                                 # (v)
    Eo, Mo = po.energies_of(L, want)
    assert np.array_equal(Eo, E2[d]) and np.array_equal(Mo, M2[d])
    og = g.observables(beta)
    oo = po.observables_of(L, E2, M2, beta, lnZ, plan["lnQ"])
    assert og["R"] == oo["R"] == R_new
    for key in OBS_KEYS:
        assert og[key] == pytest.approx(oo[key], rel=REL, abs=1e-300), (key, og[key], oo[key])
    if hist is not None:
        g.hist_accumulate(beta)
        po.hist_fold_of(L, E2, lnZ, beta, hist[0], hist[1])
        po.mag_fold_of(L, E2, M2, hist[2], hist[3])
    return og, lnZ


def plain_step(g, wl, beta_prev, beta, lnZ_ref, hist=None):
    """One temperature step on the device alone; the oracle only tracks ln Z and the histogram sums from the E vector."""
    E, _ = g.energies()
    plan = po.resample_plan(wl.R, E, wl.seed, g.resample_counter, beta - beta_prev)
    assert g.resample(beta_prev, beta) == plan["R_new"]
    g.sweep(beta, wl.theta)
    og = g.observables(beta)
    lnZ = lnZ_ref + plan["lnQ"]
    if hist is not None:
        E2, M2 = g.energies()
        g.hist_accumulate(beta)
        po.hist_fold_of(wl.L, E2, lnZ, beta, hist[0], hist[1])
        po.mag_fold_of(wl.L, E2, M2, hist[2], hist[3])
    return og, lnZ


def _check_initial(g, wl, rng, n_slots):
    """a0 at full size: sampled slots against the oracle's INIT stream (an Oracle of the sampled prefix is the
    same stream because INIT is keyed by (site, slot)), closed forms at beta = 0 on the full vectors."""
    R, N = wl.R, wl.N
    assert g.population == R and g.capacity == po.capacity(R)
    n = min(R, 2048)
    small = po.Oracle(wl.L, n, wl.seed)
    if n % 32 == 0 or n == R:
        assert np.array_equal(g.get_spins(0, n), small.get_spins())
    E, M = g.energies()
    d = _sample(rng, R, n_slots, always=(0, R - 1))
    Eo, Mo = po.energies_of(wl.L, _bits(g.get_spins_at(d)))
    assert np.array_equal(Eo, E[d]) and np.array_equal(Mo, M[d])
    # closed forms for i.i.d. spins: <E> = 0, Var E = 2N, <M^2> = N; 5 sigma of the sample mean
    assert abs(E.mean()) < 5.0 * np.sqrt(2.0 * N / R)
    assert abs(E.astype(np.float64).var() / (2.0 * N) - 1.0) < 5.0 * np.sqrt(2.0 / R)
    assert abs((M.astype(np.float64) ** 2).mean() / N - 1.0) < 5.0 * np.sqrt(2.0 / R)
    assert np.all((E + 2 * N) % 4 == 0)


def _run_fixed_schedule(cfg, checked, n_slots, last_step, rng_mode=po.RNG_PHILOX, whole=True, kinds=None):
    wl = CONFIGS[cfg]
    rng = np.random.default_rng(1000 + cfg)
    g = pa.Population(wl.L, wl.R, wl.seed)
    g.set_rng_mode(rng_mode)                                   # pa.PA_RNG_* and po.RNG_* are the same numbers (0, 1)
    _check_initial(g, wl, rng, n_slots)
    betas = wl.betas()
    lnZ = wl.N * np.log(2.0)
    assert g.lnZ == pytest.approx(lnZ, rel=1e-15)
    last = len(betas) - 1 if (RUN_ALL and whole) else last_step
    for i in range(1, last + 1):
        if i in checked:
            og, lnZ = checked_step(g, wl, betas[i - 1], betas[i], rng, n_slots, lnZ, rng_mode=rng_mode)
        else:
            og, lnZ = plain_step(g, wl, betas[i - 1], betas[i], lnZ)
        if kinds is not None:                                  # (bits that must be set, bits that must be clear) of pa_last_sweep_kind
            assert g.last_sweep_kind & kinds[0] == kinds[0] and g.last_sweep_kind & kinds[1] == 0, (i, g.last_sweep_kind)
        # population size stays close to R: every r_j is a Bernoulli rounding, sd <= sqrt(R)/2 per step
        assert abs(og["R"] - wl.R) < 8.0 * np.sqrt(wl.R)
    g.close()
    return og


def test_config2_full_size_sampled():
    """BASELINE.json configs[1] (the bench.py default): L=64, R=20000, 200 equal steps to beta=1, theta=10, seed 2.  The whole
    schedule on the device; steps 1, 2, 3, 88 (next to beta_c), 120 and 200 are checked on 1024 sampled slots each (the first
    steps are also compared in full by test_parity_gpu.py::test_config2_first_steps)."""
    og = _run_fixed_schedule(2, checked={1, 2, 3, 88, 120, 200}, n_slots=1024, last_step=200)
    assert og["beta"] == 1.0 and og["absm"] > 0.99


def test_config3_full_size_sampled():
    """BASELINE.json configs[2]: L=64, R=131072 bit-packed, 200 equal steps to beta=1, theta=10, seed 3.
    The whole schedule runs on the device (0.7 s); steps 1, 2, 88 (beta = 0.44, next to beta_c), 150 and 200 are checked."""
    og = _run_fixed_schedule(3, checked={1, 2, 88, 150, 200}, n_slots=1024, last_step=200, kinds=(pa.PA_SWEEP_RAN_COL, pa.PA_SWEEP_RAN_P64))
    assert og["beta"] == 1.0 and og["absm"] > 0.99              # ordered phase at beta = 1


def test_config5_full_size_sampled():
    """BASELINE.json configs[4]: L=256, R=10^6 (8.2 GB of packed spins, twice for the copy buffer), 500 steps of 0.001 to
    beta = 0.5, past beta_c = 0.4407.  The whole schedule runs on the device; steps 1, 2, 3, 12, then 250,
    then 438 ... 444 (beta_c, strong resampling: parents span many source groups on 4-CTA clusters), then 498, 499, 500 are
    checked on 256 sampled slots each (the oracle sweeps 256 x 65536 x 10 spins per checked step); every other step has its
    R_new recomputed by the oracle from the full E vector.  PA_FULLSIZE_STEPS=short: the first 12 steps."""
    free, _ = torch.cuda.mem_get_info()
    if free < 20 * 2**30:
        pytest.skip("needs 17 GB of device memory")
    checked = {1, 2, 3, 12, 250} | set(range(438, 445)) | {498, 499, 500}
    og = _run_fixed_schedule(5, checked=checked, n_slots=256, last_step=12)
    if RUN_ALL:
        assert og["beta"] == 0.5 and og["absm"] > 0.85                  # ordered side of beta_c


def test_config3_full_size_sampled_lcg_stream():
    """configs[2] with the paper's LCG-assisted sweep stream (O11, L236-L241): the whole schedule on the device, the same
    sampled checks; ordered at beta = 1."""
    assert pa.PA_RNG_LCG == po.RNG_LCG
    # 4096 groups >= 24 rounds of the SMs at L = 64: every sweep of this run must have taken the p = 64 (uint2) kernel by itself
    og = _run_fixed_schedule(3, checked={1, 2, 88, 200}, n_slots=1024, last_step=200, rng_mode=po.RNG_LCG,
                             kinds=(pa.PA_SWEEP_RAN_COL | pa.PA_SWEEP_RAN_P64, 0))
    assert og["beta"] == 1.0 and og["absm"] > 0.99


@pytest.mark.parametrize("side", [-1, +1])
def test_lcg_p64_gate_both_sides_equal_the_p32_bytes(side, monkeypatch):
    """The automatic choice of the p = 64 LCG kernel (L = 64, one CTA per group, a uniform launch of at least 24 rounds of the
    SMs; Table 1 L200/L204 are the p = 64 rows): one group below and one above the gate, an odd number of groups and a
    ragged last one.  Whichever kernel is taken, the bytes are those of PA_LCG_P64=0 -- through the single calls and through
    pa_anneal (whose grid covers the capacity) -- and pa_last_sweep_kind tells which one ran."""
    monkeypatch.delenv("PA_LCG_P64", raising=False)
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    G = 24 * n_sm + side                                         # odd (24 n_sm is even): the last pair of the uint2 kernel is half empty
    R = 32 * G - 5
    betas = [0.0, 0.2, 0.41]
    words = []
    for p64 in (None, 0):
        a, b = pa.Population(64, R, 64064), pa.Population(64, R, 64064)
        for x in (a, b):
            x.set_rng_mode(pa.PA_RNG_LCG)
            x.set_switch("PA_LCG_P64", p64)
            x.sweep(0.0, 1)                                      # exactly G groups: the gate itself
        assert bool(a.last_sweep_kind & pa.PA_SWEEP_RAN_P64) == (p64 is None and side > 0), (side, p64, a.last_sweep_kind)
        pa_driver.run_fixed(a, betas, 2)
        b.observables(betas[0]); b.anneal(betas, 2)
        assert a.population == b.population
        if p64 == 0:
            assert not (a.last_sweep_kind | b.last_sweep_kind) & pa.PA_SWEEP_RAN_P64
        words.append((a.get_words().tobytes(), b.get_words().tobytes()))
        a.close(); b.close()
    assert words[0][0] == words[0][1] == words[1][0] == words[1][1]


def test_config5_full_size_sampled_lcg_stream():
    """configs[4] (L=256: clusters of CTAs, quad-row walk) with the LCG-assisted stream: the whole 500-step schedule with the
    checked-step set of the Philox run (bench.py publishes a cfg5 figure for this stream).  PA_FULLSIZE_STEPS=short: 6 steps."""
    free, _ = torch.cuda.mem_get_info()
    if free < 20 * 2**30:
        pytest.skip("needs 17 GB of device memory")
    checked = {1, 2, 3, 6, 12, 250} | set(range(438, 445)) | {498, 499, 500}
    og = _run_fixed_schedule(5, checked=checked, n_slots=192, last_step=6, rng_mode=po.RNG_LCG)
    if RUN_ALL:
        assert og["beta"] == 0.5 and og["absm"] > 0.85


@pytest.mark.parametrize("mode", [0, 1])
def test_config3_whole_runs_against_kaufman(mode):
    """The whole method at full size against what the mathematics fixes ("a wealth of exact ... results"): three
    complete cfg3 runs (L=64, R=131072, 200 steps, theta=10; one pa_anneal call each) per sweep stream against Kaufman's exact
    finite-lattice e, C and beta F / N.  With R = 131072 the statistical error is ~1e-5 in e, so the bounds below are set by the
    method's own equilibration bias next to beta_c (theta = 10 at L = 64), not by noise: 3e-4 in e (3e-3 within 0.03 of beta_c),
    1.5 % in C (3 % near beta_c), 1e-4 in beta F / N -- several times the deviations measured in round 1, orders of magnitude
    below what a wrong acceptance rule, a dropped bond or a biased resampling would produce."""
    from oracle import exact_ising as ex
    wl = CONFIGS[3]
    betas = wl.betas()
    runs = []
    for seed in (11, 12, 13):
        g = pa.Population(wl.L, wl.R, seed)
        g.set_rng_mode(mode)
        g.observables(betas[0])
        runs.append(g.anneal(betas, wl.theta))
        g.close()
    for i in (20, 60, 84, 88, 92, 120, 200):
        k = ex.kaufman(betas[i], wl.L)
        near = abs(betas[i] - 0.4407) < 0.03
        e = np.mean([r[i - 1]["e"] for r in runs]); c = np.mean([r[i - 1]["C"] for r in runs]); f = np.mean([r[i - 1]["betaF_per_N"] for r in runs])
        assert abs(e - k["e"]) < (3e-3 if near else 3e-4), (betas[i], e, k["e"])
        assert abs(c - k["C"]) < (0.03 if near else 0.015) * k["C"], (betas[i], c, k["C"])
        assert abs(f - k["betaF_per_N"]) < 1e-4, (betas[i], f, k["betaF_per_N"])
        assert all(abs(r[i - 1]["R"] - wl.R) < 8 * np.sqrt(wl.R) for r in runs)
    # ordered phase: |m| -> 1, and S/N -> ln 2 / N-ish small; entropy non-negative all along
    assert all(r[-1]["absm"] > 0.99 for r in runs) and all(o["S_per_N"] > -1e-6 for r in runs for o in r)


def test_config4_full_size_adaptive_multihistogram():
    """BASELINE.json configs[3]: L=128, R=100000, adaptive steps at overlap 0.85, multi-histogram over all beta, seed 4: the
    WHOLE adaptive run to beta = 1 (about 400 steps; PA_FULLSIZE_STEPS=short: 24).  EVERY step's adaptive dbeta is recomputed
    by the oracle from the device's full E vector (41 overlap evaluations, O10) and must agree bit for bit, as must the
    realised overlap; sampled-slot checks (i)-(v) at steps 1, 2, 3, 20, the first step past every 0.1 in beta, the three steps
    around beta_c = 0.4407, and the last one; the Eq. 9 sums and the reweighted curves of the whole run at the end."""
    wl = CONFIGS[4]
    rng = np.random.default_rng(1004)
    g = pa.Population(wl.L, wl.R, wl.seed)
    _check_initial(g, wl, rng, 512)
    N = wl.N
    hist = (np.zeros(N + 1, dtype=np.int64), np.full(N + 1, -np.inf), np.zeros(N + 1, dtype=np.int64), np.zeros(N + 1, dtype=np.int64))
    lnZ = N * np.log(2.0)
    beta = wl.beta0
    E, M = g.energies()
    g.observables(beta); g.hist_accumulate(beta)
    po.hist_fold_of(wl.L, E, lnZ, beta, hist[0], hist[1])
    po.mag_fold_of(wl.L, E, M, hist[2], hist[3])
    n_steps = 100000 if RUN_ALL else 24
    checked = {1, 2, 3, 20, n_steps}
    marks = [0.1 * k for k in range(1, 10)] + [0.4407 - 1e-9]           # first step past each mark is checked in full
    around_bc = 0
    i = 0
    min_margin = float("inf")
    while beta < wl.beta_f and i < n_steps:
        i += 1
        E, _ = g.energies()
        d_g = g.adapt_dbeta(wl.target_overlap, beta, wl.beta_f)
        d_o = po.adapt_dbeta_of(wl.R, E, wl.target_overlap, beta, wl.beta_f)
        assert d_g == d_o, (i, d_g, d_o)
        assert 0.0 < d_g <= wl.beta_f - beta
        min_margin = min(min_margin, g.adapt_margins()[0])
        if i <= 60:                                                      # tripwire: all 41 decisions by exact evaluation beside the filter
            g.set_switch("PA_ADAPT_EXACT", 1)
            assert g.adapt_dbeta(wl.target_overlap, beta, wl.beta_f) == d_g and g.adapt_stats()[0] in (1, 41)
            g.set_switch("PA_ADAPT_EXACT", None)
        assert g.overlap(d_g) == po.overlap_of(wl.R, E, d_g) >= wl.target_overlap
        new = wl.beta_f if beta + d_g >= wl.beta_f else beta + d_g
        crossed = [m for m in marks if beta < m <= new]
        if any(abs(m - 0.4407) < 1e-6 for m in crossed):
            around_bc = 2                                                # this step and the next two
            checked.add(i)
        elif around_bc > 0:
            around_bc -= 1
            checked.add(i)
        if crossed:
            checked.add(i)
        if i in checked or new == wl.beta_f:
            og, lnZ = checked_step(g, wl, beta, new, rng, 512, lnZ, hist)
        else:
            og, lnZ = plain_step(g, wl, beta, new, lnZ, hist)
        beta = new
    assert i >= 20
    if RUN_ALL:
        assert beta == wl.beta_f and 100 < i < 5000 and og["absm"] > 0.99
    # the rounding bound of the histogram filter is a first-order argument: its measured safety factor
    max_err = g.adapt_margins()[1]
    print(f"adaptive filter over {i} steps: smallest |alpha' - alpha*| / threshold at a decision of the filter = {min_margin:.4g} (> 1 by "
          f"construction); largest |alpha' - alpha_exact| / first-order bound at a hand-back = {max_err:.4g} (the threshold is 4)")
    assert min_margin > 1.0 and 0.0 <= max_err < 4.0
    Hg, Dg = g.histogram()
    assert np.array_equal(Hg, hist[0])                             # integer counts: bit-exact
    fin = np.isfinite(hist[1])
    assert np.array_equal(np.isfinite(Dg), fin)
    assert np.allclose(Dg[fin], hist[1][fin], rtol=REL, atol=0)
    A1, A2 = g.mag_sums()                                          # O14: exact integers
    assert np.array_equal(A1, hist[2]) and np.array_equal(A2, hist[3])
    # O12 + O14 at full size: the reweighted curves from the device's sums against the oracle's from its own
    grid = np.linspace(0.0, beta, 25)
    rg = g.reweight(grid)
    ro = {**po.reweight_of(wl.L, hist[0], hist[1], grid), **po.reweight_mag_of(wl.L, hist[0], hist[1], hist[2], hist[3], grid)}
    for k in ("lnZ", "e", "C", "absm", "m2"):
        assert np.allclose(rg[k], ro[k], rtol=REL, atol=1e-300), k
    g.close()
