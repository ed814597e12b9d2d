"""ctypes binding of the CPU oracle (oracle/pa_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's CPU legs (cpu_baseline, --impl reference)
may import this module.  It imports nothing from paper_1703_03676_b200.
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None


class Obs(C.Structure):
    _fields_ = [("beta", C.c_double), ("e", C.c_double), ("C", C.c_double), ("absm", C.c_double),
                ("m2", C.c_double), ("m4", C.c_double), ("betaF_per_N", C.c_double),
                ("S_per_N", C.c_double), ("lnQ", C.c_double), ("R", C.c_int64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        L = _lib
        vp, i32, i64, u32, u64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_uint32, C.c_uint64, C.c_double
        L.ora_philox4x32_10.argtypes = [vp, vp, vp]; L.ora_philox4x32_10.restype = None
        L.ora_threshold.argtypes = [dbl]; L.ora_threshold.restype = u32
        L.ora_thresholds.argtypes = [dbl, vp, vp]; L.ora_thresholds.restype = None
        L.ora_tree1024.argtypes = [vp, i64]; L.ora_tree1024.restype = dbl
        L.ora_capacity.argtypes = [i64]; L.ora_capacity.restype = i64
        L.ora_sweep_slots.argtypes = [i32, u64, u32, dbl, i32, i64, vp, vp]; L.ora_sweep_slots.restype = i32
        L.ora_sweep_slots_mode.argtypes = [i32, u64, u32, dbl, i32, i64, vp, vp, i32]; L.ora_sweep_slots_mode.restype = i32
        L.ora_lcg_next.argtypes = [u32]; L.ora_lcg_next.restype = u32
        L.ora_set_rng_mode.argtypes = [vp, i32]; L.ora_set_rng_mode.restype = i32
        L.ora_energies_of.argtypes = [i32, i64, vp, vp, vp]; L.ora_energies_of.restype = i32
        L.ora_resample_plan.argtypes = [i64, i64, vp, u64, u32, dbl, vp, vp, vp, vp, vp, vp]
        L.ora_resample_plan.restype = i32
        L.ora_overlap_of.argtypes = [i64, i64, vp, dbl]; L.ora_overlap_of.restype = dbl
        L.ora_adapt_dbeta_of.argtypes = [i64, i64, vp, dbl, dbl, dbl, vp]; L.ora_adapt_dbeta_of.restype = i32
        L.ora_observables_of.argtypes = [i32, i64, vp, vp, dbl, dbl, dbl, vp]; L.ora_observables_of.restype = i32
        L.ora_hist_fold_of.argtypes = [i32, i64, vp, dbl, dbl, vp, vp]; L.ora_hist_fold_of.restype = i32
        L.ora_reweight_of.argtypes = [i32, vp, vp, i32, vp, vp, vp, vp]; L.ora_reweight_of.restype = i32
        L.ora_reweight.argtypes = [vp, i32, vp, vp, vp, vp]; L.ora_reweight.restype = i32
        L.ora_reweight_mag_of.argtypes = [i32, vp, vp, vp, vp, i32, vp, vp, vp]; L.ora_reweight_mag_of.restype = i32
        L.ora_mag_fold_of.argtypes = [i32, i64, vp, vp, vp, vp]; L.ora_mag_fold_of.restype = i32
        L.ora_get_mag_sums.argtypes = [vp, vp, vp]; L.ora_get_mag_sums.restype = i32
        L.ora_reweight_mag.argtypes = [vp, i32, vp, vp, vp]; L.ora_reweight_mag.restype = i32
        L.ora_set_couplings.argtypes = [vp, vp, vp]; L.ora_set_couplings.restype = i32
        L.ora_level_offset.argtypes = [vp]; L.ora_level_offset.restype = i32
        L.ora_sweep_slots_j.argtypes = [i32, u64, u32, dbl, i32, i64, vp, vp, i32, vp, vp]; L.ora_sweep_slots_j.restype = i32
        L.ora_energies_of_j.argtypes = [i32, i64, vp, vp, vp, vp, vp]; L.ora_energies_of_j.restype = i32
        L.ora_weighted_average.argtypes = [i32, vp, vp, i32, vp, vp]; L.ora_weighted_average.restype = i32
        L.ora_create.argtypes = [i32, i64, u64, vp]; L.ora_create.restype = i32
        L.ora_create_box.argtypes = [i32, vp, i64, u64, vp]; L.ora_create_box.restype = i32
        L.ora_num_levels.argtypes = [vp]; L.ora_num_levels.restype = i32
        L.ora_thresholds3.argtypes = [dbl, vp, vp, vp]; L.ora_thresholds3.restype = None
        L.ora_sweep_slots_3d.argtypes = [vp, u64, u32, dbl, i32, i64, vp, vp]; L.ora_sweep_slots_3d.restype = i32
        L.ora_energies_of_3d.argtypes = [vp, i64, vp, vp, vp]; L.ora_energies_of_3d.restype = i32
        L.ora_destroy.argtypes = [vp]; L.ora_destroy.restype = None
        L.ora_population.argtypes = [vp]; L.ora_population.restype = i64
        L.ora_capacity_of.argtypes = [vp]; L.ora_capacity_of.restype = i64
        L.ora_sweep_counter.argtypes = [vp]; L.ora_sweep_counter.restype = u32
        L.ora_resample_counter.argtypes = [vp]; L.ora_resample_counter.restype = u32
        L.ora_lnZ.argtypes = [vp]; L.ora_lnZ.restype = dbl
        L.ora_sweep.argtypes = [vp, dbl, i32]; L.ora_sweep.restype = i32
        L.ora_energies.argtypes = [vp, vp, vp]; L.ora_energies.restype = i32
        L.ora_resample.argtypes = [vp, dbl, dbl, vp]; L.ora_resample.restype = i32
        L.ora_adapt_dbeta.argtypes = [vp, dbl, dbl, dbl, vp]; L.ora_adapt_dbeta.restype = i32
        L.ora_overlap.argtypes = [vp, dbl, vp]; L.ora_overlap.restype = i32
        L.ora_observables.argtypes = [vp, dbl, vp]; L.ora_observables.restype = i32
        L.ora_hist_accumulate.argtypes = [vp, dbl]; L.ora_hist_accumulate.restype = i32
        L.ora_get_histogram.argtypes = [vp, vp, vp]; L.ora_get_histogram.restype = i32
        L.ora_get_spins.argtypes = [vp, i64, i64, vp]; L.ora_get_spins.restype = i32
        L.ora_set_spins.argtypes = [vp, i64, i64, vp]; L.ora_set_spins.restype = i32
        L.ora_get_resample_debug.argtypes = [vp, vp, vp, vp, vp]; L.ora_get_resample_debug.restype = i32
        L.ora_num_threads.argtypes = []; L.ora_num_threads.restype = i32
        L.ora_set_num_threads.argtypes = [i32]; L.ora_set_num_threads.restype = None
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


# ---- stateless pieces --------------------------------------------------------------------

def philox4x32_10(ctr, key):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32); key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    lib().ora_philox4x32_10(_p(ctr), _p(key), _p(out))
    return out


def threshold(p):
    return int(lib().ora_threshold(float(p)))


def thresholds(beta):
    t4, t8 = C.c_uint32(), C.c_uint32()
    lib().ora_thresholds(float(beta), C.byref(t4), C.byref(t8))
    return t4.value, t8.value


def tree1024(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return float(lib().ora_tree1024(_p(a), a.size))


def capacity(R):
    return int(lib().ora_capacity(int(R)))


RNG_PHILOX, RNG_LCG = 0, 1      # O1: one Philox number per spin; O11: Philox-seeded LCG per word


def sweep_slots(L, seed, t0, beta, theta, slot_ids, spins01, rng_mode=RNG_PHILOX):
    """theta sweeps of the replicas spins01[n][N] (uint8 0/1) living in slots slot_ids; in place."""
    slot_ids = np.ascontiguousarray(slot_ids, dtype=np.int64)
    assert spins01.dtype == np.uint8 and spins01.flags.c_contiguous
    _check(lib().ora_sweep_slots_mode(L, seed, t0, float(beta), theta, slot_ids.size, _p(slot_ids), _p(spins01),
                                      int(rng_mode)), "sweep_slots")
    return spins01


def sweep_slots_j(L, seed, t0, beta, theta, slot_ids, spins01, Jx, Jy, rng_mode=RNG_PHILOX):
    """O15: as sweep_slots, with bimodal couplings Jx, Jy (int8 [N], +-1)."""
    slot_ids = np.ascontiguousarray(slot_ids, dtype=np.int64)
    Jx = np.ascontiguousarray(Jx, dtype=np.int8); Jy = np.ascontiguousarray(Jy, dtype=np.int8)
    assert spins01.dtype == np.uint8 and spins01.flags.c_contiguous and Jx.size == L * L == Jy.size
    _check(lib().ora_sweep_slots_j(L, seed, t0, float(beta), theta, slot_ids.size, _p(slot_ids), _p(spins01), int(rng_mode),
                                   _p(Jx), _p(Jy)), "sweep_slots_j")
    return spins01


def energies_of_j(L, spins01, Jx, Jy):
    spins01 = np.ascontiguousarray(spins01, dtype=np.uint8)
    Jx = np.ascontiguousarray(Jx, dtype=np.int8); Jy = np.ascontiguousarray(Jy, dtype=np.int8)
    n = spins01.shape[0]
    E = np.empty(n, dtype=np.int32); M = np.empty(n, dtype=np.int32)
    _check(lib().ora_energies_of_j(L, n, _p(spins01), _p(Jx), _p(Jy), _p(E), _p(M)), "energies_of_j")
    return E, M


def thresholds3(beta):
    """O16: (T4, T8, T12) of the simple-cubic lattice."""
    t4, t8, t12 = C.c_uint32(), C.c_uint32(), C.c_uint32()
    lib().ora_thresholds3(float(beta), C.byref(t4), C.byref(t8), C.byref(t12))
    return t4.value, t8.value, t12.value


def sweep_slots_3d(dims, seed, t0, beta, theta, slot_ids, spins01):
    """O16: theta sweeps of the replicas spins01[n][Lx*Ly*Lz] (uint8 0/1, site = (z*Ly + y)*Lx + x) living in slots slot_ids; in place."""
    d = np.ascontiguousarray(dims, dtype=np.int32)
    slot_ids = np.ascontiguousarray(slot_ids, dtype=np.int64)
    assert d.size == 3 and spins01.dtype == np.uint8 and spins01.flags.c_contiguous and spins01.shape[1] == int(d.prod())
    _check(lib().ora_sweep_slots_3d(_p(d), seed, t0, float(beta), theta, slot_ids.size, _p(slot_ids), _p(spins01)), "sweep_slots_3d")
    return spins01


def energies_of_3d(dims, spins01):
    d = np.ascontiguousarray(dims, dtype=np.int32)
    spins01 = np.ascontiguousarray(spins01, dtype=np.uint8)
    n = spins01.shape[0]
    E = np.empty(n, dtype=np.int32); M = np.empty(n, dtype=np.int32)
    _check(lib().ora_energies_of_3d(_p(d), n, _p(spins01), _p(E), _p(M)), "energies_of_3d")
    return E, M


def lcg_next(r):
    return int(lib().ora_lcg_next(int(r)))


def energies_of(L, spins01):
    spins01 = np.ascontiguousarray(spins01, dtype=np.uint8)
    n = spins01.shape[0]
    E = np.empty(n, dtype=np.int32); M = np.empty(n, dtype=np.int32)
    _check(lib().ora_energies_of(L, n, _p(spins01), _p(E), _p(M)), "energies_of")
    return E, M


def resample_plan(R_target, E, seed, k, dbeta):
    E = np.ascontiguousarray(E, dtype=np.int32)
    R = E.size
    W = C.c_double(); R_new = C.c_int64(); lnQ = C.c_double()
    w = np.empty(R, dtype=np.float64); r = np.empty(R, dtype=np.uint32); o = np.empty(R, dtype=np.uint32)
    _check(lib().ora_resample_plan(R_target, R, _p(E), seed, k, float(dbeta), C.byref(W), _p(w), _p(r), _p(o),
                                   C.byref(R_new), C.byref(lnQ)), "resample_plan")
    return {"W": W.value, "w": w, "r": r, "o": o, "R_new": R_new.value, "lnQ": lnQ.value}


def overlap_of(R_target, E, dbeta):
    E = np.ascontiguousarray(E, dtype=np.int32)
    return float(lib().ora_overlap_of(R_target, E.size, _p(E), float(dbeta)))


def adapt_dbeta_of(R_target, E, target, beta, beta_max):
    E = np.ascontiguousarray(E, dtype=np.int32)
    d = C.c_double()
    _check(lib().ora_adapt_dbeta_of(R_target, E.size, _p(E), float(target), float(beta), float(beta_max), C.byref(d)),
           "adapt_dbeta_of")
    return d.value


def observables_of(L, E, M, beta, lnZ, lnQ):
    E = np.ascontiguousarray(E, dtype=np.int32); M = np.ascontiguousarray(M, dtype=np.int32)
    o = Obs()
    _check(lib().ora_observables_of(L, E.size, _p(E), _p(M), float(beta), float(lnZ), float(lnQ), C.byref(o)),
           "observables_of")
    return o.as_dict()


def hist_fold_of(L, E, lnZ, beta, Hsum, lnD):
    """Fold the energy histogram of E at beta into Hsum (int64[N+1]) and lnD (float64[N+1]), in place."""
    E = np.ascontiguousarray(E, dtype=np.int32)
    assert Hsum.dtype == np.int64 and lnD.dtype == np.float64 and Hsum.size == L * L + 1 == lnD.size
    _check(lib().ora_hist_fold_of(L, E.size, _p(E), float(lnZ), float(beta), _p(Hsum), _p(lnD)), "hist_fold_of")


def set_num_threads(n):
    lib().ora_set_num_threads(int(n))


def num_threads():
    return int(lib().ora_num_threads())


def reweight_of(L, Hsum, lnD, betas):
    """O12 (Sec. 2.4): lnZ, e, C at every beta from the accumulated Eq. 9 sums."""
    Hsum = np.ascontiguousarray(Hsum, dtype=np.int64); lnD = np.ascontiguousarray(lnD, dtype=np.float64)
    betas = np.ascontiguousarray(betas, dtype=np.float64)
    lnZ = np.empty(betas.size); e = np.empty(betas.size); Cv = np.empty(betas.size)
    _check(lib().ora_reweight_of(L, _p(Hsum), _p(lnD), betas.size, _p(betas), _p(lnZ), _p(e), _p(Cv)), "reweight_of")
    return {"lnZ": lnZ, "e": e, "C": Cv}


def reweight_mag_of(L, Hsum, lnD, A1, A2, betas):
    """O14: <|m|>, <m^2> at every beta from the Eq. 9 sums and the microcanonical magnetisation sums."""
    Hsum = np.ascontiguousarray(Hsum, dtype=np.int64); lnD = np.ascontiguousarray(lnD, dtype=np.float64)
    A1 = np.ascontiguousarray(A1, dtype=np.int64); A2 = np.ascontiguousarray(A2, dtype=np.int64)
    betas = np.ascontiguousarray(betas, dtype=np.float64)
    a = np.empty(betas.size); q = np.empty(betas.size)
    _check(lib().ora_reweight_mag_of(L, _p(Hsum), _p(lnD), _p(A1), _p(A2), betas.size, _p(betas), _p(a), _p(q)), "reweight_mag_of")
    return {"absm": a, "m2": q}


def mag_fold_of(L, E, M, A1, A2):
    E = np.ascontiguousarray(E, dtype=np.int32); M = np.ascontiguousarray(M, dtype=np.int32)
    assert A1.dtype == np.int64 and A2.dtype == np.int64
    _check(lib().ora_mag_fold_of(L, E.size, _p(E), _p(M), _p(A1), _p(A2)), "mag_fold_of")


def weighted_average(lnZ, A):
    """O13 (Eq. 6-7): A[M][nobs] -> (A~[nobs], omega[M])."""
    lnZ = np.ascontiguousarray(lnZ, dtype=np.float64); A = np.ascontiguousarray(A, dtype=np.float64)
    M = lnZ.size
    A = A.reshape(M, -1)
    out = np.empty(A.shape[1]); w = np.empty(M)
    _check(lib().ora_weighted_average(M, _p(lnZ), _p(A), A.shape[1], _p(out), _p(w)), "weighted_average")
    return out, w


# ---- the population handle -----------------------------------------------------------------

class Oracle:
    """The same calls as include/pa.h (pa_create, pa_sweep, ...), on the CPU oracle."""

    def __init__(self, L, R, seed, dims=None):
        """L x L square lattice, or (dims = (Lx, Ly, Lz), L ignored) a periodic simple-cubic box (O16)."""
        h = C.c_void_p()
        if dims is None:
            self.L, self.N, self.dims = L, L * L, (L, L)
            _check(lib().ora_create(L, R, seed, C.byref(h)), "create")
        else:
            d = np.ascontiguousarray(dims, dtype=np.int32)
            self.L, self.N, self.dims = int(d[0]), int(d.prod()), tuple(int(v) for v in d)
            _check(lib().ora_create_box(d.size, _p(d), R, seed, C.byref(h)), "create_box")
        self.R_target, self.seed = R, seed
        self._h = h
        self.nlev = int(lib().ora_num_levels(h)) - 1         # energies lie on -2 nlev + 4m + e0, m = 0..nlev

    @classmethod
    def box(cls, dims, R, seed):
        return cls(dims[0], R, seed, dims=dims)

    def close(self):
        if self._h:
            lib().ora_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def population(self):
        return int(lib().ora_population(self._h))

    @property
    def capacity(self):
        return int(lib().ora_capacity_of(self._h))

    @property
    def sweep_counter(self):
        return int(lib().ora_sweep_counter(self._h))

    @property
    def resample_counter(self):
        return int(lib().ora_resample_counter(self._h))

    @property
    def lnZ(self):
        return float(lib().ora_lnZ(self._h))

    def reweight(self, betas):
        betas = np.ascontiguousarray(betas, dtype=np.float64)
        lnZ = np.empty(betas.size); e = np.empty(betas.size); Cv = np.empty(betas.size)
        _check(lib().ora_reweight(self._h, betas.size, _p(betas), _p(lnZ), _p(e), _p(Cv)), "reweight")
        return {"lnZ": lnZ, "e": e, "C": Cv}

    def mag_sums(self):
        A1 = np.empty(self.nlev + 1, dtype=np.int64); A2 = np.empty(self.nlev + 1, dtype=np.int64)
        _check(lib().ora_get_mag_sums(self._h, _p(A1), _p(A2)), "get_mag_sums")
        return A1, A2

    def reweight_mag(self, betas):
        betas = np.ascontiguousarray(betas, dtype=np.float64)
        a = np.empty(betas.size); q = np.empty(betas.size)
        _check(lib().ora_reweight_mag(self._h, betas.size, _p(betas), _p(a), _p(q)), "reweight_mag")
        return {"absm": a, "m2": q}

    def set_couplings(self, Jx, Jy):
        """O15: bimodal couplings (int8 [N], +-1; Jx[s]: bond to the right of s, Jy[s]: bond below s); None, None = ferromagnet."""
        if Jx is None:
            _check(lib().ora_set_couplings(self._h, None, None), "set_couplings")
            return
        Jx = np.ascontiguousarray(Jx, dtype=np.int8); Jy = np.ascontiguousarray(Jy, dtype=np.int8)
        assert Jx.size == self.N == Jy.size
        _check(lib().ora_set_couplings(self._h, _p(Jx), _p(Jy)), "set_couplings")

    @property
    def level_offset(self):
        return int(lib().ora_level_offset(self._h))

    def set_rng_mode(self, mode):
        _check(lib().ora_set_rng_mode(self._h, int(mode)), "set_rng_mode")

    def sweep(self, beta, theta):
        _check(lib().ora_sweep(self._h, float(beta), int(theta)), "sweep")

    def energies(self):
        R = self.population
        E = np.empty(R, dtype=np.int32); M = np.empty(R, dtype=np.int32)
        _check(lib().ora_energies(self._h, _p(E), _p(M)), "energies")
        return E, M

    def resample(self, beta, beta_new):
        Rn = C.c_int64()
        rc = lib().ora_resample(self._h, float(beta), float(beta_new), C.byref(Rn))
        _check(rc, "resample")
        return Rn.value

    def resample_rc(self, beta, beta_new):
        Rn = C.c_int64()
        return lib().ora_resample(self._h, float(beta), float(beta_new), C.byref(Rn)), Rn.value

    def adapt_dbeta(self, target, beta, beta_max):
        d = C.c_double()
        _check(lib().ora_adapt_dbeta(self._h, float(target), float(beta), float(beta_max), C.byref(d)), "adapt")
        return d.value

    def overlap(self, dbeta):
        a = C.c_double()
        _check(lib().ora_overlap(self._h, float(dbeta), C.byref(a)), "overlap")
        return a.value

    def observables(self, beta):
        o = Obs()
        _check(lib().ora_observables(self._h, float(beta), C.byref(o)), "observables")
        return o.as_dict()

    def hist_accumulate(self, beta):
        _check(lib().ora_hist_accumulate(self._h, float(beta)), "hist_accumulate")

    def histogram(self):
        H = np.empty(self.nlev + 1, dtype=np.int64); D = np.empty(self.nlev + 1, dtype=np.float64)
        _check(lib().ora_get_histogram(self._h, _p(H), _p(D)), "get_histogram")
        return H, D

    def get_spins(self, j0=0, nrep=None):
        nrep = self.population - j0 if nrep is None else nrep
        out = np.empty((nrep, self.N), dtype=np.int8)
        _check(lib().ora_get_spins(self._h, j0, nrep, _p(out)), "get_spins")
        return out

    def set_spins(self, j0, spins_pm1):
        s = np.ascontiguousarray(spins_pm1, dtype=np.int8)
        _check(lib().ora_set_spins(self._h, j0, s.shape[0], _p(s)), "set_spins")

    def resample_debug(self, R_prev):
        W = C.c_double()
        w = np.empty(R_prev, dtype=np.float64); r = np.empty(R_prev, dtype=np.uint32); o = np.empty(R_prev, dtype=np.uint32)
        _check(lib().ora_get_resample_debug(self._h, C.byref(W), _p(w), _p(r), _p(o)), "resample_debug")
        return {"W": W.value, "w": w, "r": r, "o": o}
