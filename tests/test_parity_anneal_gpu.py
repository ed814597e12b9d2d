"""pa_anneal (n temperature steps without host round trips; population size and E_min resident on the device) against
(a) the same sequence of pa_resample / pa_sweep / pa_observables calls on the device: every number identical, and
(b) the CPU oracle: spins, energies, copy numbers bit-exact, observables 1e-9 (-m gpu)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("no CUDA device", allow_module_level=True)

from oracle import pa_oracle as po                      # noqa: E402
from paper_1703_03676_b200 import pa                    # noqa: E402
from paper_1703_03676_b200.workloads import CONFIGS, random_couplings     # noqa: E402
import pa_driver                                        # noqa: E402

REL = 1e-9
KEYS = ("beta", "e", "C", "absm", "m2", "m4", "betaF_per_N", "S_per_N", "lnQ", "R")


def _state(g):
    E, M = g.energies()
    return g.population, g.sweep_counter, g.resample_counter, g.lnZ, g.get_spins().tobytes(), E.tobytes(), M.tobytes()


@pytest.mark.parametrize("L,R,mode,theta,chunk", [(16, 1000, 0, 3, None), (8, 33, 1, 2, "2"), (64, 2500, 1, 2, "3"), (64, 700, 0, 1, None),
                                                   (128, 200, 0, 1, "1"), (6, 1, 0, 2, None), (32, 5000, 0, 0, None),
                                                   (64, 5300, 0, 1, None), (64, 5300, 1, 2, "3")])      # mixed launch (whole groups + lane-split tail) over the capacity-sized grid
def test_anneal_equals_step_by_step_calls_and_oracle(monkeypatch, L, R, mode, theta, chunk):
    if chunk:
        monkeypatch.setenv("PA_ANNEAL_CHUNK", chunk)                  # several chunks: tables and snapshots are re-staged
    else:
        monkeypatch.delenv("PA_ANNEAL_CHUNK", raising=False)
    betas = [0.0, 0.05, 0.12, 0.12, 0.3, 0.44, 0.6, 0.95]              # uneven steps, one of them empty (dbeta = 0)
    a, b, o = pa.Population(L, R, 41), pa.Population(L, R, 41), po.Oracle(L, R, 41)
    for x in (a, b, o):
        x.set_rng_mode(mode)
    obs_a = a.anneal(betas, theta)
    obs_b = pa_driver.run_fixed(b, betas, theta)[1:]
    obs_o = pa_driver.run_fixed(o, betas, theta)[1:]
    assert len(obs_a) == len(betas) - 1
    for x, y, z in zip(obs_a, obs_b, obs_o):
        for k in KEYS:
            assert x[k] == y[k], (k, x[k], y[k])                        # the same host arithmetic on the same device sums
            assert x[k] == pytest.approx(z[k], rel=REL, abs=1e-300), (k, x[k], z[k])
    assert _state(a) == _state(b)
    assert np.array_equal(a.get_spins(), o.get_spins())
    # the handle carries on: last resample's vectors, further single calls, a second anneal
    da, db = a.resample_debug(obs_a[-2]["R"]), b.resample_debug(obs_b[-2]["R"])
    assert da["W"] == db["W"] and np.array_equal(da["r"], db["r"]) and np.array_equal(da["o"], db["o"]) and np.array_equal(da["w"], db["w"])
    assert a.adapt_dbeta(0.8, betas[-1], 2.0) == b.adapt_dbeta(0.8, betas[-1], 2.0)
    more = [betas[-1], 1.0, 1.1]
    a.resample(more[0], more[1]); a.sweep(more[1], 1); x1 = a.observables(more[1])
    y1 = b.anneal(more[:2], 1)[0]
    assert all(x1[k] == y1[k] for k in KEYS)
    assert _state(a) == _state(b)


@pytest.mark.parametrize("cfg,nsteps,mode", [(3, 12, 0), (3, 12, 1), (5, 3, 0)])
def test_anneal_at_full_size_equals_single_calls(cfg, nsteps, mode):
    """BASELINE.json configs[2] / configs[4] at full size (capacity-sized grids, several waves, L = 256 on clusters): the packed
    population, energies and every observable after pa_anneal equal those of the single calls (which the sampled full-size
    tests tie to the oracle)."""
    wl = CONFIGS[cfg]
    free, _ = torch.cuda.mem_get_info()
    if free < 4.5 * wl.groups * wl.N * 4 + 2**30:
        pytest.skip("not enough device memory for two populations")
    betas = wl.betas()[:nsteps + 1]
    a = pa.Population(wl.L, wl.R, wl.seed); a.set_rng_mode(mode)
    obs_a = a.anneal(betas, wl.theta)
    Ea, Ma = a.energies(device=True)
    wa = torch.from_numpy(a.get_words()) if cfg != 5 else None
    R_a, lnZ_a = a.population, a.lnZ
    sample = a.get_spins_at(np.arange(0, R_a, max(1, R_a // 64), dtype=np.int64))
    if cfg == 5:
        a.close()                                                       # 16 GB each: one population at a time
    b = pa.Population(wl.L, wl.R, wl.seed); b.set_rng_mode(mode)
    obs_b = pa_driver.run_fixed(b, betas, wl.theta)[1:]
    assert obs_a == obs_b and (R_a, lnZ_a) == (b.population, b.lnZ)
    Eb, Mb = b.energies(device=True)
    assert torch.equal(Ea, Eb) and torch.equal(Ma, Mb)
    assert np.array_equal(sample, b.get_spins_at(np.arange(0, R_a, max(1, R_a // 64), dtype=np.int64)))
    if wa is not None:
        assert torch.equal(wa, torch.from_numpy(b.get_words()))


def test_anneal_with_couplings_and_histogram_between_calls():
    L, R, theta = 16, 800, 2
    Jx, Jy = random_couplings(L, 3)
    a, o = pa.Population(L, R, 5), po.Oracle(L, R, 5)
    a.set_couplings(Jx, Jy); o.set_couplings(Jx, Jy)
    betas = [0.1 * i for i in range(11)]
    a.observables(0.0); a.hist_accumulate(0.0)
    o.observables(0.0); o.hist_accumulate(0.0)
    for i in range(0, 10, 5):                                            # two anneal calls of 5 steps, a histogram fold after each
        obs = a.anneal(betas[i:i + 6], theta)
        a.hist_accumulate(betas[i + 5])
        for s in range(i + 1, i + 6):
            o.resample(betas[s - 1], betas[s]); o.sweep(betas[s], theta)
            oo = o.observables(betas[s])
            for k in KEYS:
                assert obs[s - i - 1][k] == pytest.approx(oo[k], rel=REL, abs=1e-300), (s, k)
        o.hist_accumulate(betas[i + 5])
    assert np.array_equal(a.get_spins(), o.get_spins())
    assert np.array_equal(a.histogram()[0], o.histogram()[0])
    assert np.allclose(a.histogram()[1][np.isfinite(o.histogram()[1])], o.histogram()[1][np.isfinite(o.histogram()[1])], rtol=REL)


def test_anneal_growing_calls_on_one_handle():
    """the pinned staging of pa_anneal is regrown when a later call needs more room than the first; the chunk
    events must survive that.  anneal(n=1), then anneal(n=12) with 16-step chunks, then n=40, against the single calls."""
    L, R, theta = 32, 3000, 2
    a, b = pa.Population(L, R, 9), pa.Population(L, R, 9)
    betas = [0.01 * i for i in range(54)]
    obs_a = a.anneal(betas[0:2], theta) + a.anneal(betas[1:14], theta) + a.anneal(betas[13:54], theta)
    obs_b = pa_driver.run_fixed(b, betas, theta)[1:]
    assert obs_a == obs_b
    assert _state(a) == _state(b)


def test_anneal_capacity_error_keeps_the_population_before_the_failing_step(monkeypatch):
    """O7 through pa_anneal.  A population of R = 2 can die out (R_cur = 3 with tau = 2/3 each and three failed roundings).  The
    seeds below are ones where the ORACLE's run of 12 steps of 0.12 dies at step 10, 3, 8, 5 (found with oracle/ alone; the
    resampling stream is the same on both sides).  After PA_ERR_CAPACITY the handle must hold exactly the state the single
    calls reach before their failing pa_resample (spins, E, counters, ln Z), obs_out must be valid up to there, and the
    handle must carry on."""
    import ctypes
    L, theta = 8, 1
    betas = [0.12 * i for i in range(13)]
    for chunk, seed, fail_at in (("1", 259, 10), ("16", 262, 3), ("3", 441, 8), ("16", 509, 5)):
        monkeypatch.setenv("PA_ANNEAL_CHUNK", chunk)
        o = po.Oracle(L, 2, seed)
        b = pa.Population(L, 2, seed)
        for k in range(1, fail_at):
            o.resample(betas[k - 1], betas[k]); o.sweep(betas[k], theta)
            b.resample(betas[k - 1], betas[k]); b.sweep(betas[k], theta)
        with pytest.raises(Exception):
            o.resample(betas[fail_at - 1], betas[fail_at])
        assert b.resample_rc(betas[fail_at - 1], betas[fail_at])[0] == pa.PA_ERR_CAPACITY
        a = pa.Population(L, 2, seed)
        nb = np.ascontiguousarray(betas, dtype=np.float64)
        out = (pa.pa_obs_t * (len(betas) - 1))()
        rc = pa.lib().pa_anneal(a._h, len(betas) - 1, pa._ptr(nb), theta, ctypes.cast(out, ctypes.c_void_p))
        assert rc == pa.PA_ERR_CAPACITY
        # the failing step has overwritten w, r, o: there are no vectors of a "last resampling step" to export until the next good one
        assert a.prev_population == 0 == b.prev_population
        assert pa.lib().pa_get_resample_debug(a._h, None, None, None, None) == pa.PA_ERR_INVALID_ARG
        assert a.resample_counter == fail_at - 1 == b.resample_counter == o.resample_counter
        assert _state(a) == _state(b)
        assert np.array_equal(a.get_spins(), o.get_spins())
        assert out[fail_at - 2].as_dict() == b.observables(betas[fail_at - 1])
        # the handle carries on: more sweeps, and the failing step again through both APIs (the same random numbers: fails again)
        a.sweep(betas[fail_at - 1], 2); b.sweep(betas[fail_at - 1], 2)
        assert _state(a) == _state(b)
        assert a.resample_rc(betas[fail_at - 1], betas[fail_at - 1])[0] == pa.lib().pa_anneal(
            b._h, 1, pa._ptr(np.array([betas[fail_at - 1]] * 2)), 0, None)
        assert _state(a) == _state(b)
        a.close(); b.close()


def test_anneal_errors():
    g = pa.Population(8, 100, 2)
    lib = pa.lib()
    b = np.array([0.0, 0.1, 0.05])
    assert lib.pa_anneal(g._h, 2, pa._ptr(b), 1, None) == pa.PA_ERR_INVALID_ARG          # decreasing beta
    assert lib.pa_anneal(g._h, 0, pa._ptr(b), 1, None) == pa.PA_ERR_INVALID_ARG
    assert lib.pa_anneal(g._h, 1, pa._ptr(b), -1, None) == pa.PA_ERR_INVALID_ARG
    assert lib.pa_anneal(g._h, 1, None, 1, None) == pa.PA_ERR_INVALID_ARG
    before = g.get_spins()
    assert lib.pa_anneal(g._h, 1, pa._ptr(np.array([0.0, 0.0])), 0, None) == pa.PA_OK     # dbeta = 0, theta = 0: identity
    assert np.array_equal(g.get_spins(), before) and g.population == 100
    # a huge step from a handful of replicas: R_new ~ R_target fits; a capacity overflow needs R_new > R + 1024: shrink first
    words = g.get_words()
    g.set_words(3, words[:1])
    rc = lib.pa_anneal(g._h, 1, pa._ptr(np.array([0.0, 0.01])), 0, None)
    assert rc == pa.PA_OK and abs(g.population - 100) <= 3                                # 3 replicas -> ~100 copies: within capacity


def test_timing_mask():
    """pa_set_timing: only the phases asked for are timed (the sweep by default); results do not depend on it."""
    outs = []
    for mask in (None, 0, 7):
        g = pa.Population(16, 300, 4)
        if mask is not None:
            g.set_timing(mask)
        g.resample(0.0, 0.1); g.sweep(0.1, 2); g.observables(0.1)
        if mask in (None, 7):
            assert g.last_sweep_ms() > 0.0
        else:
            with pytest.raises(pa.PaError):
                g.last_sweep_ms()
        if mask == 7:
            t, c = g.last_resample_ms()
            assert t >= c > 0.0 and g.last_measure_ms() > 0.0
        else:
            with pytest.raises(pa.PaError):
                g.last_resample_ms()
            with pytest.raises(pa.PaError):
                g.last_measure_ms()
        outs.append(g.get_spins().tobytes())
    assert outs[0] == outs[1] == outs[2]
    assert pa.lib().pa_set_timing(g._h, 8) == pa.PA_ERR_INVALID_ARG


def test_pipe_calibration_matches_the_roofline_model():
    """pa_calibrate: the integer-pipe rates bench.py's roofline rests on, re-measured -- LOP3 at 64 and
    IMAD.WIDE.U32 at 32 thread-instructions per clock per SM, the Philox round mix (2 wide multiplies + 2 LOP3) at 64."""
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    want = {0: 64.0, 1: 32.0, 2: 64.0}
    for kind, lanes in want.items():
        g, mhz = pa.pa_calibrate(kind)
        got = g * 1e3 / (mhz * sms)
        assert 1000.0 < mhz < 2500.0
        assert 0.9 * lanes < got < 1.03 * lanes, (kind, got, mhz)


def test_two_handles_interleaved_are_independent():
    """One handle = one population on its own stream, no global state (include/pa.h): two populations advanced in an
    interleaved order, give the bytes of the same
    populations advanced alone."""
    def alone(L, R, seed, mode):
        g = pa.Population(L, R, seed); g.set_rng_mode(mode)
        pa_driver.run_fixed(g, [0.0, 0.2, 0.4], 2)
        return g.get_spins().tobytes(), g.lnZ
    want_a, want_b = alone(32, 700, 1, 0), alone(64, 300, 2, 1)
    a, b = pa.Population(32, 700, 1), pa.Population(64, 300, 2)
    b.set_rng_mode(1)
    a.observables(0.0); b.observables(0.0)
    for lo, hi in ((0.0, 0.2), (0.2, 0.4)):
        a.resample(lo, hi); b.resample(lo, hi)
        b.sweep(hi, 2); a.sweep(hi, 2)
        a.observables(hi); b.observables(hi)
    assert (a.get_spins().tobytes(), a.lnZ) == want_a
    assert (b.get_spins().tobytes(), b.lnZ) == want_b


@pytest.mark.parametrize("L,R", [(16, 1000), (64, 777), (256, 40), (6, 33)])
def test_workspace_guard_bands_stay_intact(L, R):
    """compute-sanitizer is not available on the GPU pool, so out-of-bounds writes are looked for directly: the caller-owned
    workspace (pa_create_ex) sits between two 1 MiB guard bands filled with a pattern; after a run that exercises every kernel
    (both sweep streams, couplings, resampling with shrinking and growing populations, pa_anneal, histogram, reweighting,
    export / import) the bands must be untouched."""
    guard = 1 << 20
    nbytes = pa.pa_workspace_bytes(L, R)
    buf = torch.full((nbytes + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda")
    h = pa.pa_create_ex(L, R, 9, buf.data_ptr() + guard, nbytes, torch.cuda.current_stream().cuda_stream)
    g = pa.Population.__new__(pa.Population)
    g.L, g.N, g.R_target, g.seed, g._torch, g._ws, g._h = L, L * L, R, 9, torch, buf, h
    Jx, Jy = random_couplings(L, 1)
    g.set_couplings(Jx, Jy)
    g.observables(0.0); g.hist_accumulate(0.0)
    g.resample(0.0, 0.3); g.sweep(0.3, 2); g.observables(0.3); g.hist_accumulate(0.3)
    g.set_rng_mode(pa.PA_RNG_LCG)
    g.anneal([0.3, 0.5, 0.9, 1.4], 2)
    g.hist_accumulate(1.4)
    words = g.get_words()
    g.set_words(min(R, 5), words[:1])                                  # shrink to a handful: the next resample grows back to ~R
    g.resample(1.4, 1.5); g.sweep(1.5, 1)
    g.adapt_dbeta(0.8, 1.5, 3.0)
    g.reweight(np.linspace(0.0, 1.5, 7)); g.get_spins(); g.energies()
    g.set_timing(7); g.resample(1.5, 1.6); g.sweep(1.6, 1); g.observables(1.6)
    torch.cuda.synchronize()
    assert bool((buf[:guard] == 0xA5).all()) and bool((buf[guard + nbytes:] == 0xA5).all())
    g.close()


@pytest.mark.parametrize("L,R,mode,theta,chunk", [(64, 6000, 0, 2, "50"), (64, 6000, 1, 2, "37"), (64, 6000, 0, 1, None), (128, 1500, 0, 1, "7"),
                                                   (16, 1000, 0, 2, "5"), (64, 3000, 0, 0, "20"), (256, 700, 0, 1, "4")])
def test_step_host_equals_single_calls_and_oracle(monkeypatch, L, R, mode, theta, chunk):
    """pa_step_host (population in pinned host buffers between steps; sweeps in chunks of groups, finished chunks copied out on a
    second stream) = pa_set_words, pa_resample, pa_sweep, pa_observables, pa_energies, pa_get_words, and = the oracle.  Chunk sizes
    that do not divide the population, the one-piece path, a geometry without range launches (L = 16) and theta = 0 included."""
    if chunk:
        monkeypatch.setenv("PA_STEP_HOST_CHUNK", chunk)
    else:
        monkeypatch.delenv("PA_STEP_HOST_CHUNK", raising=False)
    betas = [0.0, 0.1, 0.3, 0.3, 0.45, 0.8]
    a, b, o = pa.Population(L, R, 43), pa.Population(L, R, 43), po.Oracle(L, R, 43)
    for x in (a, b, o):
        x.set_rng_mode(mode)
    Gcap = (a.capacity + 31) // 32
    wa = torch.zeros((Gcap, L * L), dtype=torch.int32, pin_memory=True)
    wb = torch.zeros((Gcap, L * L), dtype=torch.int32, pin_memory=True)
    Ea = torch.zeros(a.capacity, dtype=torch.int32, pin_memory=True)
    Ma = torch.zeros(a.capacity, dtype=torch.int32, pin_memory=True)
    a.get_words(wa)
    wb.copy_(wa)
    Ra = Rb = a.population
    for i in range(1, len(betas)):
        oa, Ra_new = a.step_host(Ra, wa, betas[i - 1], betas[i], theta, wa, Ea, Ma)
        b.set_words(Rb, wb)
        Rb_new = b.resample(betas[i - 1], betas[i])
        b.sweep(betas[i], theta)
        ob = b.observables(betas[i])
        Eb, Mb = b.energies()
        b.get_words(wb)
        assert o.resample(betas[i - 1], betas[i]) == Rb_new == Ra_new == a.population
        o.sweep(betas[i], theta)
        oo = o.observables(betas[i])
        Ga = (Ra_new + 31) // 32
        assert torch.equal(wa[:Ga], wb[:Ga]), i
        assert np.array_equal(Ea[:Ra_new].numpy(), Eb) and np.array_equal(Ma[:Ra_new].numpy(), Mb)
        Eo, Mo = o.energies()
        assert np.array_equal(Eb, Eo) and np.array_equal(Mb, Mo)
        for k in KEYS:
            assert oa[k] == ob[k], (k, oa[k], ob[k])
            assert oa[k] == pytest.approx(oo[k], rel=REL, abs=1e-300), k
        assert a.sweep_counter == b.sweep_counter == o.sweep_counter and a.lnZ == b.lnZ
        Ra = Rb = Ra_new
    assert np.array_equal(a.get_spins(), o.get_spins())


def test_environment_switches_give_the_same_bytes(monkeypatch):
    """Every tuning / fallback switch of DESIGN.md Sec. 13 that no other test sets: the same run (single calls, then pa_anneal) with
    the switch set gives the bytes and observables of the default path, which equals the oracle."""
    switches = ("PA_PDL", "PA_SMALL_PLAN", "PA_FUSE_COPY", "PA_SNAP_HOST", "PA_LCG_NOR", "PA_SWEEP_SMEM_KB", "PA_SWEEP_CMP")
    cases = [((16, 1000, 0), [{}, {"PA_PDL": "0"}, {"PA_SMALL_PLAN": "0"}, {"PA_FUSE_COPY": "0"}, {"PA_SNAP_HOST": "0"},
                              {"PA_SMALL_PLAN": "0", "PA_SNAP_HOST": "0", "PA_PDL": "0"}]),
             ((64, 700, 1), [{}, {"PA_LCG_NOR": "0"}, {"PA_LCG_NOR": "2"}, {"PA_LCG_NOR": "6"}, {"PA_LCG_NOR": "8"}, {"PA_PDL": "0"}]),
             ((128, 100, 0), [{}, {"PA_SWEEP_SMEM_KB": "32"}, {"PA_SWEEP_CMP": "2"}, {"PA_SNAP_HOST": "0"}])]
    betas = [0.0, 0.1, 0.25, 0.25, 0.45, 0.7]
    for (L, R, mode), envs in cases:
        o = po.Oracle(L, R, 47); o.set_rng_mode(mode)
        obs_o = pa_driver.run_fixed(o, betas[:4], 2)[1:]
        o_mid = o.get_spins().tobytes()
        ref = None
        for env in envs:
            for k in switches:
                monkeypatch.delenv(k, raising=False)
            for k, v in env.items():
                monkeypatch.setenv(k, v)
            g = pa.Population(L, R, 47); g.set_rng_mode(mode)
            obs = pa_driver.run_fixed(g, betas[:4], 2)[1:]
            mid = g.get_spins().tobytes()
            obs += g.anneal(betas[3:], 2)
            out = (mid, _state(g), repr(obs))
            if ref is None:
                ref = out
                assert mid == o_mid
                for a, b in zip(obs[:3], obs_o):
                    for k in KEYS:
                        assert a[k] == pytest.approx(b[k], rel=REL, abs=1e-300), k
            else:
                assert out == ref, (L, env)


def test_step_host_errors_leave_the_handle_usable():
    """pa_step_host: device buffers, a negative theta, a decreasing beta and a population size outside [1, R_cap] are refused with
    PA_ERR_INVALID_ARG before anything is touched; a step that would empty the population returns PA_ERR_CAPACITY, leaves the
    uploaded population in the handle and words_out untouched."""
    L, R = 8, 40
    g = pa.Population(L, R, 5)
    Gc = (g.capacity + 31) // 32
    w = torch.zeros((Gc, L * L), dtype=torch.int32, pin_memory=True)
    g.get_words(w)
    before = g.get_spins().copy()
    dev = w.cuda()
    for args in ((R, dev, 0.0, 0.1, 1, w), (R, w, 0.0, 0.1, 1, dev), (R, w, 0.0, 0.1, -1, w), (R, w, 0.2, 0.1, 1, w),
                 (0, w, 0.0, 0.1, 1, w), (g.capacity + 1, w, 0.0, 0.1, 1, w)):
        with pytest.raises(pa.PaError) as e:
            g.step_host(*args)
        assert e.value.code == pa.PA_ERR_INVALID_ARG
    assert np.array_equal(g.get_spins(), before) and g.population == R and g.sweep_counter == 0
    # one replica and a huge step: tau < 1 for ... a single replica always has tau = 1, so take two replicas with different energies
    g2 = pa.Population(4, 2, 1)
    o2 = po.Oracle(4, 2, 1)
    w2 = torch.zeros(((g2.capacity + 31) // 32, 16), dtype=torch.int32, pin_memory=True)
    g2.get_words(w2)
    out = torch.full_like(w2, 0x5a5a5a5a)
    died = False
    beta = 0.0
    for k in range(40):                                   # strong steps until the oracle's population dies out (or 40 steps pass)
        try:
            o2.resample(beta, beta + 2.0)
        except Exception:
            died = True
            with pytest.raises(pa.PaError) as e:
                g2.step_host(g2.population, w2, beta, beta + 2.0, 1, out)
            assert e.value.code == pa.PA_ERR_CAPACITY
            assert torch.all(out == 0x5a5a5a5a)
            assert np.array_equal(g2.get_spins(), o2.get_spins()) and g2.population == o2.population
            break
        o2.sweep(beta + 2.0, 1)
        _, Rn = g2.step_host(g2.population, w2, beta, beta + 2.0, 1, w2)
        assert Rn == o2.population and np.array_equal(g2.get_spins(), o2.get_spins())
        beta += 2.0
    assert died or g2.population == o2.population
