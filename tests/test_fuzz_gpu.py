"""Seeded differential fuzz of the CUDA path against the CPU oracle (-m gpu): random lattice sizes (any even L, so the generic and
the column-walk kernels, one CTA and clusters), ragged population sizes, both sweep streams, ferromagnet and random +-J couplings,
uneven temperature schedules with very large steps (empty and many-fold copy numbers, parents spanning many source groups),
single calls and pa_anneal.  Spins, energies, copy numbers: bit-exact; observables: 1e-9."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("no CUDA device", allow_module_level=True)

from oracle import pa_oracle as po                      # noqa: E402
from paper_1703_03676_b200 import pa                    # noqa: E402
from paper_1703_03676_b200.workloads import random_couplings     # noqa: E402

REL = 1e-9
KEYS = ("beta", "e", "C", "absm", "m2", "m4", "betaF_per_N", "S_per_N", "lnQ", "R")


def _case(i):
    rng = np.random.default_rng(90000 + i)
    L = int(rng.choice([4, 6, 8, 10, 12, 14, 16, 20, 24, 32, 40, 48, 64, 64, 96, 128]))
    R = int(rng.choice([1, 2, 31, 32, 33, 63, 65, 100, 257, 500, 1023, 1025, 2000]))
    if L >= 96:
        R = min(R, 300)
    mode = int(rng.integers(0, 2))
    coupl = bool(rng.integers(0, 2))
    theta = int(rng.choice([0, 1, 1, 2, 3]))
    n = int(rng.integers(2, 6))
    steps = rng.choice([0.0, 0.01, 0.05, 0.2, 0.6, 1.5], size=n, p=[0.1, 0.2, 0.3, 0.2, 0.15, 0.05])
    betas = np.concatenate([[0.0], np.cumsum(steps)]).tolist()
    api = "anneal" if rng.integers(0, 2) else "steps"
    return L, R, 1000 + i, mode, coupl, theta, betas, api


@pytest.mark.parametrize("i", range(int(os.environ.get("PA_FUZZ_N", "48"))))       # PA_FUZZ_N=2000 for a long hunt
def test_random_case(i):
    L, R, seed, mode, coupl, theta, betas, api = _case(i)
    g, o = pa.Population(L, R, seed), po.Oracle(L, R, seed)
    g.set_rng_mode(mode); o.set_rng_mode(mode)
    if coupl:
        Jx, Jy = random_couplings(L, seed)
        g.set_couplings(Jx, Jy); o.set_couplings(Jx, Jy)
    # the oracle first: a tiny population can die out (all copy numbers 0: PA_ERR_CAPACITY, O7) -- then the device must say so too
    oo, dead_at = [], None
    for k in range(1, len(betas)):
        try:
            o.resample(betas[k - 1], betas[k])
        except Exception:
            dead_at = k
            break
        o.sweep(betas[k], theta)
        oo.append(o.observables(betas[k]))
    if dead_at is not None:
        g.observables(betas[0])
        if api == "anneal":
            with pytest.raises(pa.PaError) as e:
                g.anneal(betas, theta)
        else:
            for k in range(1, dead_at):
                g.resample(betas[k - 1], betas[k]); g.sweep(betas[k], theta)
            with pytest.raises(pa.PaError) as e:
                g.resample(betas[dead_at - 1], betas[dead_at])
        assert e.value.code == pa.PA_ERR_CAPACITY
        # both APIs: the population is the one before the failing step, the steps before it have been applied (O7)
        assert g.population == o.population and g.sweep_counter == o.sweep_counter and g.resample_counter == o.resample_counter
        assert g.lnZ == pytest.approx(o.lnZ, rel=1e-12)
        assert np.array_equal(g.get_spins(), o.get_spins()), i
        Eg, Mg = g.energies(); Eo, Mo = o.energies()
        assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
        return
    og = []
    if api == "anneal":
        g.observables(betas[0])
        og = g.anneal(betas, theta)
    else:
        o2 = po.Oracle(L, R, seed); o2.set_rng_mode(mode)
        if coupl:
            o2.set_couplings(Jx, Jy)
        for k in range(1, len(betas)):
            R_prev = o2.population
            o2.resample(betas[k - 1], betas[k]); o2.sweep(betas[k], theta)
            g.resample(betas[k - 1], betas[k])
            a, b = g.resample_debug(R_prev), o2.resample_debug(R_prev)
            assert a["W"] == b["W"] and np.array_equal(a["r"], b["r"]) and np.array_equal(a["o"], b["o"]), (i, k)
            g.sweep(betas[k], theta)
            og.append(g.observables(betas[k]))
            assert np.array_equal(g.get_spins(), o2.get_spins()), (i, k)
    for a, b in zip(og, oo):
        for key in KEYS:
            assert a[key] == pytest.approx(b[key], rel=REL, abs=1e-300), (i, key, a[key], b[key])
    assert g.population == o.population and g.sweep_counter == o.sweep_counter and g.resample_counter == o.resample_counter
    assert np.array_equal(g.get_spins(), o.get_spins()), i
    Eg, Mg = g.energies(); Eo, Mo = o.energies()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    g.hist_accumulate(betas[-1]); o.hist_accumulate(betas[-1])
    assert np.array_equal(g.histogram()[0], o.histogram()[0])
    for x, y in zip(g.mag_sums(), o.mag_sums()):
        assert np.array_equal(x, y)


def _run_pair(g, o, betas, theta, api, tag):
    """Advance both through the schedule (single calls or one pa_anneal call) and compare everything."""
    oo = []
    for k in range(1, len(betas)):
        o.resample(betas[k - 1], betas[k]); o.sweep(betas[k], theta)
        oo.append(o.observables(betas[k]))
    if api == "anneal":
        g.observables(betas[0])
        og = g.anneal(betas, theta)
    elif api == "host":
        Gc = (g.capacity + 31) // 32
        w = torch.zeros((Gc, g.N), dtype=torch.int32, pin_memory=True)
        g.get_words(w)
        og, Rh = [], g.population
        for k in range(1, len(betas)):
            ob, Rh = g.step_host(Rh, w, betas[k - 1], betas[k], theta, w)
            og.append(ob)
    else:
        og = []
        for k in range(1, len(betas)):
            g.resample(betas[k - 1], betas[k]); g.sweep(betas[k], theta)
            og.append(g.observables(betas[k]))
    for a, b in zip(og, oo):
        for key in KEYS:
            assert a[key] == pytest.approx(b[key], rel=REL, abs=1e-300), (tag, key, a[key], b[key])
    assert g.population == o.population and g.sweep_counter == o.sweep_counter and g.resample_counter == o.resample_counter
    assert np.array_equal(g.get_spins(), o.get_spins()), tag
    Eg, Mg = g.energies(); Eo, Mo = o.energies()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo), tag


@pytest.mark.parametrize("i", range(int(os.environ.get("PA_FUZZ_BOX_N", "16"))))
def test_random_box_case(i):
    """The same differential fuzz on random periodic boxes (O16): even edges from 2 (double bonds) to 16, cubes of 8 and 16 (the
    column-walk sweep and quad-column energy kernels) and boxes with three different edges (the any-edge kernels), ragged
    populations, single calls / pa_anneal / pa_step_host."""
    rng = np.random.default_rng(70000 + i)
    if rng.integers(0, 3) == 0:
        e = int(rng.choice([8, 16])); dims = (e, e, e)
    else:
        dims = tuple(int(v) for v in rng.choice([2, 4, 6, 8, 10, 12, 16], size=3))
    R = int(rng.choice([1, 31, 33, 100, 257, 700]))
    if np.prod(dims) >= 2048:
        R = min(R, 100)
    theta = int(rng.choice([1, 1, 2, 3]))
    steps = rng.choice([0.0, 0.01, 0.05, 0.1, 0.3], size=int(rng.integers(2, 5)), p=[0.1, 0.25, 0.35, 0.2, 0.1])
    betas = np.concatenate([[0.0], np.cumsum(steps)]).tolist()
    api = str(rng.choice(["steps", "anneal", "host"]))
    o = po.Oracle.box(dims, R, 500 + i)
    try:
        probe = po.Oracle.box(dims, R, 500 + i)
        for k in range(1, len(betas)):
            probe.resample(betas[k - 1], betas[k]); probe.sweep(betas[k], theta)
    except Exception:
        pytest.skip("the population dies out on this schedule (covered by test_random_case)")
    g = pa.Population.box(dims, R, 500 + i)
    _run_pair(g, o, betas, theta, api, (i, dims, R, api))


@pytest.mark.parametrize("i", range(int(os.environ.get("PA_FUZZ_MEDIUM_N", "6"))))
def test_random_medium_case(i):
    """Medium populations on the column-walk kernels: random sizes around whole rounds of the 148 SMs (the mixed launch of whole
    groups plus lane-quarter CTAs, its capacity-sized grid inside pa_anneal, the chunked sweeps of pa_step_host), both streams."""
    rng = np.random.default_rng(80000 + i)
    L = int(rng.choice([64, 64, 128]))
    rounds = int(rng.integers(1, 3)) if L == 64 else 1
    R = 32 * 148 * rounds + int(rng.integers(-40, 1500))
    mode = int(rng.integers(0, 2))
    theta = int(rng.choice([1, 2]))
    betas = [0.0, 0.2, 0.2 + float(rng.choice([0.05, 0.25]))]
    api = str(rng.choice(["steps", "anneal", "host"]))
    if api == "host":
        os.environ["PA_STEP_HOST_CHUNK"] = str(int(rng.choice([37, 60, 148])))
    try:
        g, o = pa.Population(L, R, 900 + i), po.Oracle(L, R, 900 + i)
        g.set_rng_mode(mode); o.set_rng_mode(mode)
        _run_pair(g, o, betas, theta, api, (i, L, R, mode, api))
    finally:
        os.environ.pop("PA_STEP_HOST_CHUNK", None)
