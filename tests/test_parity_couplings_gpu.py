"""GPU parity of the bimodal-coupling workload (O15) against the CPU oracle (-m gpu): spins, energies,
copy numbers and histogram counts bit-exact, fp64 observables and reweighted curves to 1e-9."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("no CUDA device", allow_module_level=True)

from oracle import pa_oracle as po                      # noqa: E402
from paper_1703_03676_b200 import pa                    # noqa: E402
import pa_driver                                        # noqa: E402

REL = 1e-9
OBS_KEYS = ("beta", "e", "C", "absm", "m2", "m4", "betaF_per_N", "S_per_N", "lnQ")


def _random_j(L, seed, odd=None):
    rng = np.random.default_rng(seed)
    Jx = (rng.integers(0, 2, L * L) * 2 - 1).astype(np.int8); Jy = (rng.integers(0, 2, L * L) * 2 - 1).astype(np.int8)
    if odd is not None and (int((Jx < 0).sum() + (Jy < 0).sum()) % 2 == 1) != odd:
        Jx[3] = -Jx[3]
    return Jx, Jy


def _same(g, o):
    assert g.population == o.population and g.sweep_counter == o.sweep_counter
    assert np.array_equal(g.get_spins(), o.get_spins())
    Eg, Mg = g.energies(); Eo, Mo = o.energies()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)


@pytest.mark.parametrize("L,R,mode", [(4, 40, 0), (6, 70, 0), (16, 200, 1), (32, 100, 0), (64, 96, 1), (128, 40, 0), (256, 33, 1), (192, 33, 0),
                                      (64, 96, 0), (128, 40, 1), (256, 33, 0), (192, 33, 1)])
def test_sweep_and_energies_with_couplings_bit_exact(L, R, mode):
    """Generic kernel (L < 64, L = 192 on clusters) and both column-walk kernels (L = 64, 128 on one CTA, L = 256 on clusters with DSMEM
    halos), both sweep streams, ragged last group."""
    Jx, Jy = _random_j(L, 100 + L)
    g, o = pa.Population(L, R, 31 + L), po.Oracle(L, R, 31 + L)
    g.set_couplings(Jx, Jy); o.set_couplings(Jx, Jy)
    g.set_rng_mode(mode); o.set_rng_mode(mode)
    assert g.level_offset == o.level_offset
    _same(g, o)                                                         # energies of the random start under J
    for beta, theta in [(0.0, 1), (0.4, 2), (1.2, 3)]:
        g.sweep(beta, theta); o.sweep(beta, theta)
        _same(g, o)
    g.set_couplings(None, None); o.set_couplings(None, None)            # back to the ferromagnet
    assert g.level_offset == 0
    g.sweep(0.5, 1); o.sweep(0.5, 1)
    _same(g, o)


@pytest.mark.parametrize("odd", [False, True])
def test_whole_run_with_couplings(odd):
    """Annealing runs on a frustrated sample (even / odd number of negative bonds = level offset 0 / 2): every step's observables,
    the final state, Eq. 9 sums, microcanonical magnetisation sums, reweighted curves, adaptive step."""
    L, R, theta = 16, 1500, 3
    Jx, Jy = _random_j(L, 7, odd=odd)
    g, o = pa.Population(L, R, 8), po.Oracle(L, R, 8)
    g.set_couplings(Jx, Jy); o.set_couplings(Jx, Jy)
    assert g.level_offset == o.level_offset == (2 if odd else 0)
    betas = [0.08 * i for i in range(16)]
    og = pa_driver.run_fixed(g, betas, theta, hist=True)
    oo = pa_driver.run_fixed(o, betas, theta, hist=True)
    for a, b in zip(og, oo):
        assert a["R"] == b["R"]
        for k in OBS_KEYS:
            assert a[k] == pytest.approx(b[k], rel=REL, abs=1e-300), (k, a[k], b[k])
    _same(g, o)
    Hg, Dg = g.histogram(); Ho, Do = o.histogram()
    assert np.array_equal(Hg, Ho)
    fin = np.isfinite(Do)
    assert np.array_equal(np.isfinite(Dg), fin) and np.allclose(Dg[fin], Do[fin], rtol=REL, atol=0)
    for a, b in zip(g.mag_sums(), o.mag_sums()):
        assert np.array_equal(a, b)
    grid = np.linspace(0.0, 1.3, 14)
    rg, ro = g.reweight(grid), {**o.reweight(grid), **o.reweight_mag(grid)}
    for k in ("lnZ", "e", "C", "absm", "m2"):
        assert np.allclose(rg[k], ro[k], rtol=REL, atol=1e-300), k
    assert g.adapt_dbeta(0.8, betas[-1], 3.0) == o.adapt_dbeta(0.8, betas[-1], 3.0)
    # couplings are frozen once a histogram exists
    assert pa.lib().pa_set_couplings(g._h, None, None) == pa.PA_ERR_INVALID_ARG


def test_gauge_invariance_on_the_device():
    """Mattis couplings J_ab = eps_a eps_b: the device trajectory is the gauge-transformed ferromagnetic device trajectory."""
    L, R = 32, 64
    rng = np.random.default_rng(5)
    eps = (rng.integers(0, 2, (L, L)) * 2 - 1).astype(np.int8)
    Jx = (eps * np.roll(eps, -1, axis=1)).reshape(-1).astype(np.int8); Jy = (eps * np.roll(eps, -1, axis=0)).reshape(-1).astype(np.int8)
    f, m = pa.Population(L, R, 77), pa.Population(L, R, 77)
    m.set_couplings(Jx, Jy)
    m.set_spins(0, (f.get_spins() * eps.reshape(1, -1)).astype(np.int8))
    assert np.array_equal(f.energies()[0], m.energies()[0])
    f.sweep(0.45, 5); m.sweep(0.45, 5)
    assert np.array_equal(m.get_spins(), f.get_spins() * eps.reshape(1, -1))
    assert np.array_equal(f.energies()[0], m.energies()[0])
    bad = Jx.copy(); bad[0] = 0
    assert pa.lib().pa_set_couplings(m._h, pa._ptr(bad), pa._ptr(Jy)) == pa.PA_ERR_INVALID_ARG
