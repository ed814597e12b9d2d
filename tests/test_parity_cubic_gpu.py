"""GPU parity of the simple-cubic lattice (pa_create_box; O16) against the CPU oracle's box mode:
spins, energies, copy numbers bit-exact at every step; observables, ln D, reweighted curves to 1e-9 (-m gpu)."""
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
KEYS = ("beta", "e", "C", "absm", "m2", "m4", "betaF_per_N", "S_per_N", "lnQ", "R")


def _bits(spins_pm1):
    return np.ascontiguousarray((spins_pm1 > 0).astype(np.uint8))


def _same_state(g, o):
    assert g.population == o.population and g.sweep_counter == o.sweep_counter and g.resample_counter == o.resample_counter
    assert np.array_equal(g.get_spins(), o.get_spins())
    Eg, Mg = g.energies(); Eo, Mo = o.energies()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)


def _obs_close(a, b):
    for k in KEYS:
        assert a[k] == pytest.approx(b[k], rel=REL, abs=1e-300), (k, a[k], b[k])


# edges of length 2 (double bonds), three different edges, one plane per CTA (clusters), ragged R, cubes
@pytest.mark.parametrize("dims,R,C", [((4, 2, 2), 100, None), ((2, 2, 2), 33, None), ((6, 4, 2), 700, None), ((6, 4, 2), 700, "2"),
                                      ((4, 4, 4), 1000, None), ((4, 4, 4), 1000, "4"), ((8, 8, 8), 300, "2"), ((8, 8, 8), 300, "8"),
                                      ((16, 16, 16), 96, None), ((16, 16, 16), 65, "4"), ((10, 6, 4), 50, "2"), ((32, 32, 32), 40, None), ((64, 64, 64), 33, None)])
def test_box_run_every_step(monkeypatch, dims, R, C):
    if C:
        monkeypatch.setenv("PA_SWEEP_C", C)
    else:
        monkeypatch.delenv("PA_SWEEP_C", raising=False)
    g, o = pa.Population.box(dims, R, 17), po.Oracle.box(dims, R, 17)
    assert g.N == o.N and g.nlev == o.nlev == 3 * g.N // 2 and g.capacity == o.capacity
    _same_state(g, o)
    betas = [0.0, 0.05, 0.12, 0.12, 0.2, 0.2216, 0.3, 0.6]
    _obs_close(g.observables(betas[0]), o.observables(betas[0]))
    g.hist_accumulate(betas[0]); o.hist_accumulate(betas[0])
    for i in range(1, len(betas)):
        R_prev = g.population
        assert g.resample(betas[i - 1], betas[i]) == o.resample(betas[i - 1], betas[i])
        a, b = g.resample_debug(R_prev), o.resample_debug(R_prev)
        assert a["W"] == b["W"] and np.array_equal(a["w"], b["w"]) and np.array_equal(a["r"], b["r"]) and np.array_equal(a["o"], b["o"])
        theta = 1 + (i % 3)
        g.sweep(betas[i], theta); o.sweep(betas[i], theta)
        _same_state(g, o)
        _obs_close(g.observables(betas[i]), o.observables(betas[i]))
        g.hist_accumulate(betas[i]); o.hist_accumulate(betas[i])
    Hg, Dg = g.histogram(); Ho, Do = o.histogram()
    assert Hg.size == g.nlev + 1 and np.array_equal(Hg, Ho)
    fin = np.isfinite(Do)
    assert np.array_equal(np.isfinite(Dg), fin) and np.allclose(Dg[fin], Do[fin], rtol=REL, atol=0)
    for x, y in zip(g.mag_sums(), o.mag_sums()):
        assert np.array_equal(x, y)
    grid = np.array([0.01, 0.1, 0.21, 0.5])
    rg, ro = g.reweight(grid), {**o.reweight(grid), **o.reweight_mag(grid)}
    for k in ("lnZ", "e", "C", "absm", "m2"):
        assert np.allclose(rg[k], ro[k], rtol=REL, atol=1e-300), k


def test_cube_generic_and_fast_index_arithmetic_agree(monkeypatch):
    """Cubes of 8 .. 64 run on the column-walk kernel (a thread walks down z; default) or, with PA_SWEEP_KIND=2, on the kernel whose
    index arithmetic is shifts and masks; PA_SWEEP_KIND=0 / PA_MEASURE_GENERIC=1 force the any-edge kernels (integer divisions).
    Same bytes, same energies, for one CTA per group and for clusters (z-neighbours over DSMEM)."""
    for L, R, C in ((8, 500, None), (8, 300, "2"), (16, 200, None), (16, 100, "4"), (32, 64, None), (32, 40, "8"), (64, 33, None)):
        out = []
        for kind in (None, "2", "0"):
            for k in ("PA_SWEEP_KIND", "PA_MEASURE_GENERIC", "PA_SWEEP_C"):
                monkeypatch.delenv(k, raising=False)
            if kind:
                monkeypatch.setenv("PA_SWEEP_KIND", kind)
            if kind == "0":
                monkeypatch.setenv("PA_MEASURE_GENERIC", "1")
            if C:
                monkeypatch.setenv("PA_SWEEP_C", C)
            g = pa.Population.box((L, L, L), R, 23)
            g.sweep(0.2, 3)
            E, M = g.energies()
            out.append((g.get_words().tobytes(), E.tobytes(), M.tobytes()))
        assert out[0] == out[1] == out[2], (L, C)


def test_box_adaptive_anneal_and_export():
    """The rest of the path on a box: adaptive step (bit-identical beta sequence), pa_anneal = single calls, spin and word
    export / import in the box's site order s = (z*Ly + y)*Lx + x."""
    dims, R = (8, 4, 6), 1500
    g, o = pa.Population.box(dims, R, 3), po.Oracle.box(dims, R, 3)
    bg, og = pa_driver.run_adaptive(g, 0.0, 0.3, 2, 0.8, hist=True, max_steps=12)
    bo, oo = pa_driver.run_adaptive(o, 0.0, 0.3, 2, 0.8, hist=True, max_steps=12)
    assert bg == bo and len(bg) > 4
    for a, b in zip(og, oo):
        _obs_close(a, b)
    _same_state(g, o)
    more = [bg[-1], bg[-1] + 0.01, bg[-1] + 0.03]
    a = g.anneal(more, 2)
    b = pa_driver.run_fixed(o, more, 2)[1:]
    for x, y in zip(a, b):
        _obs_close(x, y)
    _same_state(g, o)
    # words: interchange layout word[g][s]; a round trip through set_words / set_spins reproduces the state
    w = g.get_words()
    sp = g.get_spins()
    N = g.N
    unpacked = ((w[:, None, :] >> np.arange(32, dtype=np.uint32)[None, :, None]) & 1).reshape(-1, N)[:g.population]
    assert np.array_equal(unpacked.astype(np.int8) * 2 - 1, sp)
    h = pa.Population.box(dims, R, 99)
    h.set_words(g.population, w)
    assert np.array_equal(h.get_spins(), sp)
    h.set_spins(5, -sp[5:40])
    chk = sp.copy(); chk[5:40] = -chk[5:40]
    assert np.array_equal(h.get_spins(), chk)
    assert np.array_equal(h.get_spins_at(np.array([0, 7, 39, 40, g.population - 1])), chk[[0, 7, 39, 40, g.population - 1]])
    E1, M1 = h.energies()
    E2, M2 = po.energies_of_3d(dims, _bits(chk))
    assert np.array_equal(E1, E2) and np.array_equal(M1, M2)


def test_box_errors():
    import ctypes as C
    lib = pa.lib()
    h, n = C.c_void_p(), C.c_size_t()
    for bad in ((3, 4, 4), (4, 4, 0), (4, 5, 4), (128, 128, 128), (64, 64, 66)):
        d = np.ascontiguousarray(bad, dtype=np.int32)
        assert lib.pa_workspace_bytes_box(3, pa._ptr(d), 100, C.byref(n)) == pa.PA_ERR_INVALID_ARG
        assert lib.pa_create_box(3, pa._ptr(d), 100, 1, None, 0, None, C.byref(h)) == pa.PA_ERR_INVALID_ARG
    d = np.ascontiguousarray((4, 4, 4), dtype=np.int32)
    assert lib.pa_create_box(4, pa._ptr(d), 100, 1, None, 0, None, C.byref(h)) == pa.PA_ERR_INVALID_ARG
    g = pa.Population.box((4, 4, 4), 64, 1)
    assert lib.pa_set_rng_mode(g._h, pa.PA_RNG_LCG) == pa.PA_ERR_INVALID_ARG
    J = np.ones(64, dtype=np.int8)
    assert lib.pa_set_couplings(g._h, pa._ptr(J), pa._ptr(J)) == pa.PA_ERR_INVALID_ARG
    nd, dd = C.c_int(), (C.c_int * 3)()
    assert lib.pa_dims(g._h, C.byref(nd), dd) == pa.PA_OK and nd.value == 3 and list(dd) == [4, 4, 4]
    sq = pa.Population(8, 64, 1)
    assert lib.pa_dims(sq._h, C.byref(nd), dd) == pa.PA_OK and nd.value == 2 and list(dd)[:2] == [8, 8]
    assert int(lib.pa_num_levels(sq._h)) == 65 and int(lib.pa_num_levels(g._h)) == 97
    # ndim = 2 through the box entry point is the square lattice
    d2 = np.ascontiguousarray((8, 8), dtype=np.int32)
    assert lib.pa_create_box(2, pa._ptr(d2), 64, 1, None, 0, None, C.byref(h)) == pa.PA_OK
    assert np.array_equal(pa_spins(h), sq.get_spins())
    lib.pa_destroy(h)


def pa_spins(h):
    out = np.empty((64, 64), dtype=np.int8)
    assert pa.lib().pa_get_spins(h, 0, 64, pa._ptr(out)) == pa.PA_OK
    return out


def test_cube_L32_full_size_sampled():
    """A production-size cube: 32^3 sites, R = 20 000 (625 groups of 128 KB, clusters of two CTAs), 6 temperature steps across the
    ordering transition; sampled slots are swept by the oracle (same slot ids and sweep counter) and the resampling plan is
    recomputed from the full E vector, as in the full-size 2D tests."""
    dims, R, theta = (32, 32, 32), 20000, 3
    N = 32768
    rng = np.random.default_rng(5)
    g = pa.Population.box(dims, R, 21)
    betas = [0.0, 0.1, 0.18, 0.2216, 0.24, 0.3, 0.5]
    lnZ = N * np.log(2.0)
    for i in range(1, len(betas)):
        E, M = g.energies()
        plan = po.resample_plan(R, E, 21, g.resample_counter, betas[i] - betas[i - 1])
        R_prev = g.population
        parent = np.repeat(np.arange(R_prev, dtype=np.int64), plan["r"])
        d = np.unique(np.concatenate([[0, 31, 32, plan["R_new"] - 1], rng.choice(plan["R_new"], 96, replace=False)]))
        pre = g.get_spins_at(parent[d])
        Eo, Mo = po.energies_of_3d(dims, _bits(pre))
        assert np.array_equal(Eo, E[parent[d]]) and np.array_equal(Mo, M[parent[d]])
        assert g.resample(betas[i - 1], betas[i]) == plan["R_new"]
        dbg = g.resample_debug(R_prev)
        assert dbg["W"] == plan["W"] and np.array_equal(dbg["r"], plan["r"]) and np.array_equal(dbg["o"], plan["o"])
        lnZ += plan["lnQ"]
        assert g.lnZ == pytest.approx(lnZ, rel=1e-13)
        post = g.get_spins_at(d)
        assert np.array_equal(post, pre)
        t0 = g.sweep_counter
        g.sweep(betas[i], theta)
        want = po.sweep_slots_3d(dims, 21, t0, betas[i], theta, d, _bits(post))
        assert np.array_equal(_bits(g.get_spins_at(d)), want)
        obs = g.observables(betas[i])
        assert abs(obs["R"] - R) < 8 * np.sqrt(R)
    # far below the ordering temperature (beta_c = 0.2217 on the infinite lattice) after a six-step quench: domains, most bonds satisfied
    assert obs["e"] < -2.0 and obs["beta"] == 0.5
