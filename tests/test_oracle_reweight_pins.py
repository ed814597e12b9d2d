"""Pins of the oracle's multi-histogram reweighting (O12; Sec. 2.4, Eq. 9) and of the
weighted averages over independent runs (O13; Sec. 2.2, Eq. 6-7), -m "not gpu".  No expected value comes
from the oracle itself or from the CUDA path."""
import math

import numpy as np
import pytest

from oracle import exact_ising as ex
from oracle import pa_oracle as po
import pa_driver


def test_reweight_exact_density_of_states_in_exact_averages_out():
    # feed the EXACT g(E) of the 4x4 torus (brute-force enumeration) as the histogram sum with unit denominators:
    # the reweighted lnZ, e, C must be the exact canonical values of the enumeration at every beta
    L, N = 4, 16
    g = ex.density_of_states(L)
    H = np.zeros(N + 1, dtype=np.int64)
    for E, c in g.items():
        H[(E + 2 * N) // 4] = c
    lnD = np.zeros(N + 1)
    betas = np.array([0.0, 0.1, 0.3, 0.4406868, 0.7, 1.0, 2.5])
    out = po.reweight_of(L, H, lnD, betas)
    for i, b in enumerate(betas):
        exact = ex.exact_small(float(b), L)
        assert out["lnZ"][i] == pytest.approx(-exact["betaF_per_N"] * N, rel=1e-12)
        assert out["e"][i] == pytest.approx(exact["e"], rel=1e-12, abs=1e-14)
        assert out["C"][i] == pytest.approx(exact["C"], rel=1e-10, abs=1e-14)
    # a common factor of the denominators shifts lnZ only: Omega -> Omega / c
    out2 = po.reweight_of(L, H, lnD + math.log(7.0), betas)
    assert np.allclose(out2["lnZ"], out["lnZ"] - math.log(7.0), rtol=0, atol=1e-12)
    assert np.allclose(out2["e"], out["e"], rtol=1e-13) and np.allclose(out2["C"], out["C"], rtol=1e-10, atol=1e-14)


def test_reweight_single_level_and_large_arguments():
    # one populated level E: Z = Omega exp(-beta E), e = E/N, C = 0 -- also where exp(-beta E) alone would overflow
    L, N = 32, 1024
    H = np.zeros(N + 1, dtype=np.int64); lnD = np.zeros(N + 1)
    H[0] = 2                                                           # the two ground states, E = -2N
    out = po.reweight_of(L, H, lnD, np.array([0.5, 400.0]))
    assert out["lnZ"][0] == pytest.approx(math.log(2) + 0.5 * 2 * N, rel=1e-14)
    assert out["lnZ"][1] == pytest.approx(math.log(2) + 400.0 * 2 * N, rel=1e-14)
    assert np.all(out["e"] == -2.0) and np.all(out["C"] == 0.0)


def _runs(L, R, betas, theta, seeds):
    out = []
    for s in seeds:
        o = po.Oracle(L, R, s)
        obs = pa_driver.run_fixed(o, betas, theta, hist=True)
        out.append((o, obs))
    return out


def test_reweight_from_pa_runs_matches_exact_L4():
    # Eq. 9 sums accumulated over a whole annealing run, then reweighted to temperatures BETWEEN the simulated
    # ones: exact enumeration values within the seed scatter
    L, R, theta = 4, 4000, 5
    betas = [i / 40 for i in range(41)]
    grid = np.array([0.0125, 0.2375, 0.44, 0.6625, 0.9875])
    runs = _runs(L, R, betas, theta, list(range(300, 316)))
    vals = {k: np.array([o.reweight(grid)[k] for o, _ in runs]) for k in ("lnZ", "e", "C")}
    for i, b in enumerate(grid):
        exact = ex.exact_small(float(b), L)
        want = {"lnZ": -exact["betaF_per_N"] * L * L, "e": exact["e"], "C": exact["C"]}
        for k in want:
            v = vals[k][:, i]
            sigma = v.std(ddof=1) / math.sqrt(len(runs))
            assert abs(v.mean() - want[k]) < 4 * sigma + 1e-12, (b, k, v.mean(), want[k], sigma)


def test_reweight_from_pa_runs_matches_kaufman_L16(cfg1_oracle_runs):
    # configs[0] of BASELINE.json: reweighted curves at off-grid temperatures against Kaufman's exact finite-L
    # results; the multi-histogram estimate also has to be at least as sharp as the single-temperature one
    L = 16
    grid = np.array([0.105, 0.305, 0.4355, 0.605, 0.955])
    _, runs = cfg1_oracle_runs
    vals = {k: np.array([o.reweight(grid)[k] for o, _ in runs]) for k in ("lnZ", "e", "C")}
    for i, b in enumerate(grid):
        k_ex = ex.kaufman(float(b), L)
        for k in ("lnZ", "e", "C"):
            v = vals[k][:, i]
            sigma = v.std(ddof=1) / math.sqrt(len(runs))
            assert abs(v.mean() - k_ex[k]) < 4 * sigma + 1e-9, (b, k, v.mean(), k_ex[k], sigma)
    # scatter of the reweighted energy at beta = 0.305 vs the scatter of the direct estimates at 0.30 and 0.31
    direct = np.array([[obs[30]["e"], obs[31]["e"]] for _, obs in runs])
    assert vals["e"][:, 1].std(ddof=1) < 1.5 * direct.std(axis=0, ddof=1).max()


# ---------------------------------------------------------------------------------------------
# O14 magnetisation reweighting from microcanonical sums (L129)
# ---------------------------------------------------------------------------------------------

def test_reweight_mag_exact_microcanonical_sums_in_exact_averages_out():
    # exact g(E) and the exact sums of |M| and M^2 over all states of each energy level (enumeration of the 4x4 torus):
    # the reweighted <|m|>, <m^2> must be the exact canonical values at every beta
    L, N = 4, 16
    E, M = ex.enumerate_states(L)
    H = np.zeros(N + 1, dtype=np.int64); A1 = np.zeros(N + 1, dtype=np.int64); A2 = np.zeros(N + 1, dtype=np.int64)
    np.add.at(H, (E + 2 * N) // 4, 1)
    np.add.at(A1, (E + 2 * N) // 4, np.abs(M))
    np.add.at(A2, (E + 2 * N) // 4, M * M)
    betas = np.array([0.0, 0.2, 0.4406868, 0.8, 2.0])
    out = po.reweight_mag_of(L, H, np.zeros(N + 1), A1, A2, betas)
    for i, b in enumerate(betas):
        exact = ex.exact_small(float(b), L)
        assert out["absm"][i] == pytest.approx(exact["absm"], rel=1e-12)
        assert out["m2"][i] == pytest.approx(exact["m2"], rel=1e-12)
    # the fold itself: |M| and M^2 land on the level of their replica's energy, exact integers
    A1f = np.zeros(N + 1, dtype=np.int64); A2f = np.zeros(N + 1, dtype=np.int64)
    po.mag_fold_of(L, E[:5000].astype(np.int32), M[:5000].astype(np.int32), A1f, A2f)
    w1 = np.zeros(N + 1, dtype=np.int64); w2 = np.zeros(N + 1, dtype=np.int64)
    np.add.at(w1, (E[:5000] + 2 * N) // 4, np.abs(M[:5000])); np.add.at(w2, (E[:5000] + 2 * N) // 4, M[:5000] ** 2)
    assert np.array_equal(A1f, w1) and np.array_equal(A2f, w2)


def test_reweight_mag_from_pa_runs_matches_exact_L4():
    L, R, theta = 4, 4000, 5
    betas = [i / 40 for i in range(41)]
    grid = np.array([0.0125, 0.2375, 0.44, 0.6625, 0.9875])
    runs = _runs(L, R, betas, theta, list(range(400, 416)))
    vals = {k: np.array([o.reweight_mag(grid)[k] for o, _ in runs]) for k in ("absm", "m2")}
    for i, b in enumerate(grid):
        exact = ex.exact_small(float(b), L)
        for k in ("absm", "m2"):
            v = vals[k][:, i]
            sigma = v.std(ddof=1) / math.sqrt(len(runs))
            assert abs(v.mean() - exact[k]) < 4 * sigma + 1e-12, (b, k, v.mean(), exact[k], sigma)
    # sum over levels of the folded sums = sum over all folded replicas (the direct observables times R N, R N^2)
    o, obs = runs[0]
    A1, A2 = o.mag_sums()
    assert A1.sum() == round(sum(x["absm"] * x["R"] * L * L for x in obs))
    assert A2.sum() == round(sum(x["m2"] * x["R"] * (L * L) ** 2 for x in obs))


# ---------------------------------------------------------------------------------------------
# O13 weighted averages over M independent runs (Eq. 6-7)
# ---------------------------------------------------------------------------------------------

def test_weighted_average_closed_forms():
    rng = np.random.default_rng(0)
    A = rng.normal(size=(5, 3))
    lnZ = rng.normal(size=5) * 3 + 700.0                               # exp(lnZ) overflows fp64: log-domain weights
    out, w = po.weighted_average(lnZ, A)
    assert abs(w.sum() - 1.0) < 1e-14 and np.all(w > 0)
    # Eq. 7 in exact rational-free form: ratios of weights = exp of free-energy differences
    for a in range(5):
        for b in range(5):
            assert w[a] / w[b] == pytest.approx(math.exp(lnZ[a] - lnZ[b]), rel=1e-12)
    assert np.allclose(out, (w[:, None] * A).sum(0), rtol=1e-14, atol=1e-15)          # Eq. 6
    # M = 1: the run itself; equal free energies: the arithmetic mean; a common shift of lnZ changes nothing
    o1, w1 = po.weighted_average(lnZ[:1], A[:1]); assert w1[0] == 1.0 and np.array_equal(o1, A[0])
    o2, w2 = po.weighted_average(np.full(5, -3.0), A); assert np.allclose(o2, A.mean(0), rtol=1e-14, atol=1e-15)
    o3, w3 = po.weighted_average(lnZ - 1234.5, A); assert np.allclose(w3, w, rtol=1e-11)
    # one run dominating by 800 e-folds takes all the weight
    o4, w4 = po.weighted_average(np.array([0.0, 800.0]), A[:2]); assert w4[1] == 1.0 and np.array_equal(o4, A[1])


def test_weighted_average_removes_the_small_population_bias_L4():
    # "by combining the data from independent runs not only statistical errors are decreased, but also
    # systematic deviations can be reduced ... if one uses weighted averages".  Tiny populations (R = 10) are
    # visibly biased; exp(lnZ_m) is an unbiased estimator of Z (Ref. [7, 9]), so (i) the mean of exp(lnZ_m - lnZ_exact)
    # is 1 and (ii) the weighted average of M = 3000 runs sits on the exact value while the plain mean does not.
    L, R, theta, M = 4, 10, 1, 3000
    betas = [0.0, 0.2, 0.4]                                            # big steps, one sweep: a strongly biased single run
    lnZ = np.empty(M); e = np.empty(M)
    for m in range(M):
        o = po.Oracle(L, R, 5000 + m)
        obs = pa_driver.run_fixed(o, betas, theta)
        lnZ[m] = -obs[-1]["betaF_per_N"] * L * L
        e[m] = obs[-1]["e"]
    exact = ex.exact_small(betas[-1], L)
    lnZ_exact = -exact["betaF_per_N"] * L * L
    ratio = np.exp(lnZ - lnZ_exact)
    assert abs(ratio.mean() - 1.0) < 5 * ratio.std(ddof=1) / math.sqrt(M)
    # blocks of 100 runs: scatter of the weighted and of the plain block means
    wb = np.array([po.weighted_average(lnZ[i:i + 100], e[i:i + 100, None])[0][0] for i in range(0, M, 100)])
    pb = np.array([e[i:i + 100].mean() for i in range(0, M, 100)])
    full, _ = po.weighted_average(lnZ, e[:, None])
    se_w = wb.std(ddof=1) / math.sqrt(len(wb))
    se_p = pb.std(ddof=1) / math.sqrt(len(pb))
    assert abs(full[0] - exact["e"]) < 5 * se_w, (full[0], exact["e"], se_w)
    assert abs(pb.mean() - exact["e"]) > 5 * se_p, (pb.mean(), exact["e"], se_p)      # the plain mean IS biased
