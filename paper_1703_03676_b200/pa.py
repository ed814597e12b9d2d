"""Thin Python binding of the C-ABI library declared in include/pa.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels behind these calls; this module computes
nothing.  PyTorch is used for device memory (the workspace tensor handed to pa_create_ex), for
the CUDA stream and for moving result vectors; there is no CPU fallback -- if the library or a
CUDA device is missing the calls raise.

The module-level functions have the names of the C entry points (pa_create, pa_sweep, ...).
`Population` wraps a handle with the same verbs (sweep, energies, resample, adapt_dbeta,
observables, hist_accumulate, ...), which is also the interface of oracle.pa_oracle.Oracle, so
that tests can drive both with one loop (tests/pa_driver.py).
"""
import ctypes as C
import os
import re

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libpa_b200.so")
HEADER = os.path.join(os.path.dirname(HERE), "include", "pa.h")

PA_OK, PA_ERR_INVALID_ARG, PA_ERR_CAPACITY, PA_ERR_CUDA, PA_ERR_WORKSPACE, PA_ERR_NOMEM = 0, -1, -2, -3, -4, -5
PA_ERR_STATIC_LIMIT = -6
PA_WAVG_STATIC_MAX_RUNS = 4096
PA_RNG_PHILOX, PA_RNG_LCG = 0, 1
PA_TIME_SWEEP, PA_TIME_RESAMPLE, PA_TIME_MEASURE = 1, 2, 4
PA_SWEEP_RAN_COL, PA_SWEEP_RAN_SPLIT, PA_SWEEP_RAN_P64, PA_SWEEP_RAN_MIXED = 1, 2, 4, 8


class PaError(RuntimeError):
    def __init__(self, code, what, detail=""):
        self.code = code
        super().__init__(f"{what}: {strerror(code)} ({code}) {detail}".strip())


class pa_obs_t(C.Structure):
    _fields_ = [("beta", C.c_double), ("e", C.c_double), ("C", C.c_double), ("absm", C.c_double),
                ("m2", C.c_double), ("m4", C.c_double), ("betaF_per_N", C.c_double),
                ("S_per_N", C.c_double), ("lnQ", C.c_double), ("R", C.c_int64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def declared_symbols():
    """Names of the functions include/pa.h declares."""
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pa_[a-z0-9_]+)\s*\(", text)))


def lib():
    """Load libpa_b200.so (building it first if the sources are newer).  Raises if it cannot be loaded."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        from . import build as _build
        _build.build()
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, u32, u64, dbl, sz = C.c_void_p, C.c_int, C.c_int64, C.c_uint32, C.c_uint64, C.c_double, C.c_size_t
    sig = {
        "pa_capacity": ([i64], i64),
        "pa_workspace_bytes": ([i32, i64, C.POINTER(sz)], i32),
        "pa_create": ([i32, i64, u64, C.POINTER(vp)], i32),
        "pa_create_ex": ([i32, i64, u64, vp, sz, vp, C.POINTER(vp)], i32),
        "pa_workspace_bytes_box": ([i32, vp, i64, C.POINTER(sz)], i32),
        "pa_create_box": ([i32, vp, i64, u64, vp, sz, vp, C.POINTER(vp)], i32),
        "pa_dims": ([vp, C.POINTER(i32), vp], i32),
        "pa_num_levels": ([vp], i64),
        "pa_destroy": ([vp], None),
        "pa_sweep": ([vp, dbl, i32], i32),
        "pa_anneal": ([vp, i32, vp, i32, vp], i32),
        "pa_set_timing": ([vp, i32], i32),
        "pa_set_rng_mode": ([vp, i32], i32),
        "pa_set_couplings": ([vp, vp, vp], i32),
        "pa_level_offset": ([vp], i32),
        "pa_get_rng_mode": ([vp], i32),
        "pa_energies": ([vp, vp, vp], i32),
        "pa_resample": ([vp, dbl, dbl, C.POINTER(i64)], i32),
        "pa_adapt_dbeta": ([vp, dbl, dbl, dbl, C.POINTER(dbl)], i32),
        "pa_overlap": ([vp, dbl, C.POINTER(dbl)], i32),
        "pa_adapt_stats": ([vp, C.POINTER(i32), C.POINTER(i32)], i32),
        "pa_observables": ([vp, dbl, C.POINTER(pa_obs_t)], i32),
        "pa_hist_accumulate": ([vp, dbl], i32),
        "pa_get_histogram": ([vp, vp, vp], i32),
        "pa_reweight": ([vp, i32, vp, vp, vp, vp, vp, vp], i32),
        "pa_get_mag_sums": ([vp, vp, vp], i32),
        "pa_weighted_average": ([i32, vp, vp, i32, vp, vp], i32),
        "pa_weighted_average_static": ([i32, vp, vp, i32, vp, vp], i32),
        "pa_weighted_average_static_max_runs": ([], i32),
        "pa_get_spins": ([vp, i64, i64, vp], i32),
        "pa_get_spins_at": ([vp, vp, i64, vp], i32),
        "pa_set_spins": ([vp, i64, i64, vp], i32),
        "pa_get_words": ([vp, vp], i32),
        "pa_set_words": ([vp, i64, vp], i32),
        "pa_step_host": ([vp, i64, vp, dbl, dbl, i32, vp, vp, vp, C.POINTER(pa_obs_t), C.POINTER(i64)], i32),
        "pa_get_resample_debug": ([vp, C.POINTER(dbl), vp, vp, vp], i32),
        "pa_population": ([vp], i64),
        "pa_prev_population": ([vp], i64),
        "pa_capacity_of": ([vp], i64),
        "pa_sweep_counter": ([vp], u32),
        "pa_resample_counter": ([vp], u32),
        "pa_lnZ": ([vp], dbl),
        "pa_set_counters": ([vp, u32, u32, dbl], i32),
        "pa_adapt_margins": ([vp, C.POINTER(dbl), C.POINTER(dbl)], i32),
        "pa_launch_count": ([vp], i64),
        "pa_last_sweep_kind": ([vp], i32),
        "pa_set_switch": ([vp, C.c_char_p, i32, i64], i32),
        "pa_last_sweep_ms": ([vp, C.POINTER(C.c_float)], i32),
        "pa_last_resample_ms": ([vp, C.POINTER(C.c_float), C.POINTER(C.c_float)], i32),
        "pa_last_measure_ms": ([vp, C.POINTER(C.c_float)], i32),
        "pa_calibrate": ([i32, C.POINTER(dbl), C.POINTER(dbl)], i32),
        "pa_strerror": ([i32], C.c_char_p),
        "pa_last_cuda_error": ([vp], C.c_char_p),
        "pa_version": ([], C.c_char_p),
    }
    for name, (args, res) in sig.items():
        f = getattr(L, name)
        f.argtypes = args
        f.restype = res
    _lib = L
    return L


def strerror(code):
    return lib().pa_strerror(int(code)).decode()


def _ptr(x):
    """A raw address for a numpy array (host) or a torch tensor (host or device); None -> NULL."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        assert x.flags.c_contiguous
        return C.c_void_p(x.ctypes.data)
    return C.c_void_p(x.data_ptr())       # torch tensor


# ---- module-level functions with the C names ------------------------------------------------

def pa_capacity(R):
    return int(lib().pa_capacity(int(R)))


def pa_workspace_bytes(L, R):
    n = C.c_size_t()
    rc = lib().pa_workspace_bytes(L, R, C.byref(n))
    if rc:
        raise PaError(rc, "pa_workspace_bytes")
    return n.value


def pa_calibrate(kind):
    g, mhz = C.c_double(), C.c_double()
    rc = lib().pa_calibrate(kind, C.byref(g), C.byref(mhz))
    if rc:
        raise PaError(rc, "pa_calibrate")
    return g.value, mhz.value


def pa_create(L, R, seed):
    h = C.c_void_p()
    rc = lib().pa_create(L, R, seed, C.byref(h))
    if rc:
        raise PaError(rc, "pa_create")
    return h


def pa_create_ex(L, R, seed, dev_ws_ptr, ws_bytes, cuda_stream):
    h = C.c_void_p()
    rc = lib().pa_create_ex(L, R, seed, C.c_void_p(dev_ws_ptr), ws_bytes, C.c_void_p(cuda_stream), C.byref(h))
    if rc:
        raise PaError(rc, "pa_create_ex")
    return h


def pa_destroy(h):
    lib().pa_destroy(h)


def pa_weighted_average(lnZ, A):
    """Sec. 2.2 (Eq. 6-7): A[M][nobs] of M independent runs with free-energy estimates lnZ[M] -> (A~[nobs], omega[M])."""
    lnZ = np.ascontiguousarray(lnZ, dtype=np.float64)
    M = lnZ.size
    A = np.ascontiguousarray(A, dtype=np.float64).reshape(M, -1)
    out = np.empty(A.shape[1]); w = np.empty(M)
    rc = lib().pa_weighted_average(M, _ptr(lnZ), _ptr(A), A.shape[1], _ptr(out), _ptr(w))
    if rc != PA_OK:
        raise PaError(rc, "pa_weighted_average")
    return out, w


def pa_weighted_average_static(d_lnZ, d_A, d_A_out, cuda_stream=None):
    """Eq. 6-7 like pa_weighted_average, for callers that must not allocate device memory (all of it is already handed
    out, or other streams must not be stalled by cudaMalloc / cudaFree, or a blocking driver call is not allowed where they
    run): the library allocates nothing, the weights live in a fixed 32 KiB array inside it.  d_lnZ [M], d_A [M, nobs] and
    d_A_out [nobs] are contiguous float64 CUDA tensors of the current device that the caller made beforehand; at most
    PA_WAVG_STATIC_MAX_RUNS runs (PaError with PA_ERR_STATIC_LIMIT beyond).  The kernel is enqueued on `cuda_stream` (a raw
    cudaStream_t value; None = torch's current stream) and the call does not wait: read d_A_out after synchronising that
    stream.  Calls on one GPU share the array: never let two of them run at the same time on different streams.  The first
    call on a device also looks the array up; make it at start-up, before any stream capture."""
    import torch
    for t in (d_lnZ, d_A, d_A_out):
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise PaError(PA_ERR_INVALID_ARG, "pa_weighted_average_static", "contiguous float64 CUDA tensors expected")
    M, nobs = d_lnZ.numel(), d_A_out.numel()
    if d_A.numel() != M * nobs:
        raise PaError(PA_ERR_INVALID_ARG, "pa_weighted_average_static", "A must hold M * nobs values")
    st = torch.cuda.current_stream().cuda_stream if cuda_stream is None else cuda_stream
    rc = lib().pa_weighted_average_static(M, _ptr(d_lnZ), _ptr(d_A) if nobs else None, nobs,
                                          _ptr(d_A_out) if nobs else None, C.c_void_p(st))
    if rc != PA_OK:
        raise PaError(rc, "pa_weighted_average_static")


class Population:
    """One population on the current CUDA device.  Workspace and stream come from PyTorch
    (pa_create_ex) unless own_memory=True (pa_create: cudaMalloc + private stream)."""

    def __init__(self, L, R, seed, stream=None, own_memory=False, dims=None):
        """L x L square lattice, or (dims = (Lx, Ly, Lz); L ignored) a periodic simple-cubic box (pa_create_box)."""
        import torch
        if not torch.cuda.is_available():
            raise PaError(PA_ERR_CUDA, "Population", "no CUDA device: this library has no CPU path")
        self._torch = torch
        self._ws = None
        self.R_target, self.seed = R, seed
        if dims is not None:
            d = np.ascontiguousarray(dims, dtype=np.int32)
            self.L, self.N, self.dims = int(d[0]), int(d.prod()), tuple(int(v) for v in d)
            h = C.c_void_p()
            if own_memory:
                rc = lib().pa_create_box(d.size, _ptr(d), R, seed, None, 0, None, C.byref(h))
            else:
                n = C.c_size_t()
                rc = lib().pa_workspace_bytes_box(d.size, _ptr(d), R, C.byref(n))
                if rc:
                    raise PaError(rc, "pa_workspace_bytes_box")
                self._ws = torch.empty(n.value, dtype=torch.uint8, device="cuda")
                self._stream = stream if stream is not None else torch.cuda.current_stream()
                rc = lib().pa_create_box(d.size, _ptr(d), R, seed, C.c_void_p(self._ws.data_ptr()), n.value,
                                         C.c_void_p(self._stream.cuda_stream), C.byref(h))
            if rc:
                raise PaError(rc, "pa_create_box")
            self._h = h
        else:
            self.L, self.N, self.dims = L, L * L, (L, L)
            if own_memory:
                self._h = pa_create(L, R, seed)
            else:
                nbytes = pa_workspace_bytes(L, R)
                self._ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
                self._stream = stream if stream is not None else torch.cuda.current_stream()
                self._h = pa_create_ex(L, R, seed, self._ws.data_ptr(), nbytes, self._stream.cuda_stream)
        self.nlev = int(lib().pa_num_levels(self._h)) - 1

    @classmethod
    def box(cls, dims, R, seed, **kw):
        return cls(dims[0], R, seed, dims=dims, **kw)

    def close(self):
        if getattr(self, "_h", None):
            pa_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        if rc:
            raise PaError(rc, what, lib().pa_last_cuda_error(self._h).decode() if rc == PA_ERR_CUDA else "")

    # scalars
    @property
    def population(self):
        return int(lib().pa_population(self._h))

    @property
    def capacity(self):
        return int(lib().pa_capacity_of(self._h))

    @property
    def sweep_counter(self):
        return int(lib().pa_sweep_counter(self._h))

    @property
    def resample_counter(self):
        return int(lib().pa_resample_counter(self._h))

    @property
    def lnZ(self):
        return float(lib().pa_lnZ(self._h))

    @property
    def launch_count(self):
        return int(lib().pa_launch_count(self._h))

    @property
    def last_sweep_kind(self):
        """PA_SWEEP_RAN_* bits of the kernel the last sweep() launched (diagnostics)."""
        return int(lib().pa_last_sweep_kind(self._h))

    def set_switch(self, name, value=None):
        """pa_set_switch: give the switch `name` (an environment variable's name, e.g. "PA_ADAPT_EXACT") the integer `value` on this
        live handle; value=None returns it to "not set".  The environment itself is read only when a handle is created."""
        self._check(lib().pa_set_switch(self._h, name.encode(), 0 if value is None else 1, 0 if value is None else int(value)), "pa_set_switch")

    def set_counters(self, t, k, lnZ):
        self._check(lib().pa_set_counters(self._h, t, k, float(lnZ)), "pa_set_counters")

    # the path
    def anneal(self, betas, theta):
        """pa_anneal: resample betas[i-1] -> betas[i], theta sweeps, measure, for i = 1..len(betas)-1, without host round trips;
        betas[0] must be the current temperature.  Returns the observables of betas[1:]."""
        betas = np.ascontiguousarray(betas, dtype=np.float64)
        n = betas.size - 1
        out = (pa_obs_t * n)()
        self._check(lib().pa_anneal(self._h, n, _ptr(betas), int(theta), C.cast(out, C.c_void_p)), "pa_anneal")
        return [o.as_dict() for o in out]

    def set_couplings(self, Jx, Jy):
        """Bimodal couplings (int8 [N], +-1; Jx[s]: bond to the right of s = y*L+x, Jy[s]: bond below); None, None = ferromagnet."""
        if Jx is None:
            self._check(lib().pa_set_couplings(self._h, None, None), "pa_set_couplings")
            return
        Jx = np.ascontiguousarray(Jx, dtype=np.int8); Jy = np.ascontiguousarray(Jy, dtype=np.int8)
        assert Jx.size == self.N == Jy.size
        self._check(lib().pa_set_couplings(self._h, _ptr(Jx), _ptr(Jy)), "pa_set_couplings")

    @property
    def level_offset(self):
        return int(lib().pa_level_offset(self._h))

    def set_rng_mode(self, mode):
        self._check(lib().pa_set_rng_mode(self._h, int(mode)), "pa_set_rng_mode")

    @property
    def rng_mode(self):
        return int(lib().pa_get_rng_mode(self._h))

    def sweep(self, beta, theta):
        self._check(lib().pa_sweep(self._h, float(beta), int(theta)), "pa_sweep")

    def energies(self, device=False):
        """(E, M) as numpy int32 arrays, or as torch cuda tensors if device=True."""
        R = self.population
        if device:
            E = self._torch.empty(R, dtype=self._torch.int32, device="cuda")
            M = self._torch.empty(R, dtype=self._torch.int32, device="cuda")
        else:
            E = np.empty(R, dtype=np.int32); M = np.empty(R, dtype=np.int32)
        self._check(lib().pa_energies(self._h, _ptr(E), _ptr(M)), "pa_energies")
        return E, M

    def energies_into(self, E, M=None):
        self._check(lib().pa_energies(self._h, _ptr(E), _ptr(M)), "pa_energies")

    def resample(self, beta, beta_new):
        Rn = C.c_int64()
        self._check(lib().pa_resample(self._h, float(beta), float(beta_new), C.byref(Rn)), "pa_resample")
        return Rn.value

    def resample_rc(self, beta, beta_new):
        Rn = C.c_int64()
        return lib().pa_resample(self._h, float(beta), float(beta_new), C.byref(Rn)), Rn.value

    def adapt_dbeta(self, target, beta, beta_max):
        d = C.c_double()
        self._check(lib().pa_adapt_dbeta(self._h, float(target), float(beta), float(beta_max), C.byref(d)), "pa_adapt_dbeta")
        return d.value

    def adapt_stats(self):
        """(exact evaluations, histogram-kernel launches) of the last adapt_dbeta."""
        a, b = C.c_int(), C.c_int()
        self._check(lib().pa_adapt_stats(self._h, C.byref(a), C.byref(b)), "pa_adapt_stats")
        return a.value, b.value

    def adapt_margins(self):
        """(min_margin of the last adapt_dbeta, max_error over the handle's life): the tripwire of pa_adapt_margins."""
        a, b = C.c_double(), C.c_double()
        self._check(lib().pa_adapt_margins(self._h, C.byref(a), C.byref(b)), "pa_adapt_margins")
        return a.value, b.value

    def overlap(self, dbeta):
        a = C.c_double()
        self._check(lib().pa_overlap(self._h, float(dbeta), C.byref(a)), "pa_overlap")
        return a.value

    def observables(self, beta):
        o = pa_obs_t()
        self._check(lib().pa_observables(self._h, float(beta), C.byref(o)), "pa_observables")
        return o.as_dict()

    def hist_accumulate(self, beta):
        self._check(lib().pa_hist_accumulate(self._h, float(beta)), "pa_hist_accumulate")

    def histogram(self):
        H = np.empty(self.nlev + 1, dtype=np.int64); D = np.empty(self.nlev + 1, dtype=np.float64)
        self._check(lib().pa_get_histogram(self._h, _ptr(H), _ptr(D)), "pa_get_histogram")
        return H, D

    def reweight(self, betas):
        """Sec. 2.4 (Eq. 9): lnZ, e, C, <|m|>, <m^2> at every beta of `betas` from the accumulated multi-histogram sums."""
        betas = np.ascontiguousarray(betas, dtype=np.float64)
        out = {k: np.empty(betas.size) for k in ("lnZ", "e", "C", "absm", "m2")}
        self._check(lib().pa_reweight(self._h, betas.size, _ptr(betas), *[_ptr(out[k]) for k in ("lnZ", "e", "C", "absm", "m2")]),
                    "pa_reweight")
        return out

    def mag_sums(self):
        A1 = np.empty(self.nlev + 1, dtype=np.int64); A2 = np.empty(self.nlev + 1, dtype=np.int64)
        self._check(lib().pa_get_mag_sums(self._h, _ptr(A1), _ptr(A2)), "pa_get_mag_sums")
        return A1, A2

    # state export / import
    def get_spins(self, j0=0, nrep=None):
        nrep = self.population - j0 if nrep is None else nrep
        out = np.empty((nrep, self.N), dtype=np.int8)
        self._check(lib().pa_get_spins(self._h, j0, nrep, _ptr(out)), "pa_get_spins")
        return out

    def get_spins_at(self, slots):
        slots = np.ascontiguousarray(slots, dtype=np.int64)
        out = np.empty((slots.size, self.N), dtype=np.int8)
        self._check(lib().pa_get_spins_at(self._h, _ptr(slots), slots.size, _ptr(out)), "pa_get_spins_at")
        return out

    def set_spins(self, j0, spins_pm1):
        s = np.ascontiguousarray(spins_pm1, dtype=np.int8)
        self._check(lib().pa_set_spins(self._h, j0, s.shape[0], _ptr(s)), "pa_set_spins")

    def get_words(self, out=None):
        if out is None:
            out = np.empty(((self.population + 31) // 32, self.N), dtype=np.uint32)
        self._check(lib().pa_get_words(self._h, _ptr(out)), "pa_get_words")
        return out

    def set_words(self, R, words):
        self._check(lib().pa_set_words(self._h, int(R), _ptr(words)), "pa_set_words")

    def step_host(self, R_in, words_in, beta, beta_new, theta, words_out, E_out=None, M_out=None):
        """pa_step_host: one temperature step with the population in host buffers; returns (observables dict, R_new)."""
        obs, Rn = pa_obs_t(), C.c_int64()
        self._check(lib().pa_step_host(self._h, int(R_in), _ptr(words_in), float(beta), float(beta_new), int(theta), _ptr(words_out),
                                       _ptr(E_out), _ptr(M_out), C.byref(obs), C.byref(Rn)), "pa_step_host")
        return obs.as_dict(), Rn.value

    @property
    def prev_population(self):
        return int(lib().pa_prev_population(self._h))

    def resample_debug(self, R_prev=None):
        """Vectors of the last successful resampling step; their length is pa_prev_population (R_prev, if given, must equal it)."""
        n = self.prev_population
        if R_prev is not None and int(R_prev) != n:
            raise PaError(PA_ERR_INVALID_ARG, "pa_get_resample_debug", f"R_prev = {R_prev}, the library's is {n}")
        R_prev = n
        W = C.c_double()
        w = np.empty(R_prev, dtype=np.float64); r = np.empty(R_prev, dtype=np.uint32); o = np.empty(R_prev, dtype=np.uint32)
        self._check(lib().pa_get_resample_debug(self._h, C.byref(W), _ptr(w), _ptr(r), _ptr(o)), "pa_get_resample_debug")
        return {"W": W.value, "w": w, "r": r, "o": o}

    # timing (CUDA events recorded by the library on its stream)
    def set_timing(self, mask):
        """Which phases record CUDA timing events (PA_TIME_* mask; default: the sweep only)."""
        self._check(lib().pa_set_timing(self._h, int(mask)), "pa_set_timing")

    def last_sweep_ms(self):
        ms = C.c_float()
        self._check(lib().pa_last_sweep_ms(self._h, C.byref(ms)), "pa_last_sweep_ms")
        return ms.value

    def last_measure_ms(self):
        ms = C.c_float()
        self._check(lib().pa_last_measure_ms(self._h, C.byref(ms)), "pa_last_measure_ms")
        return ms.value

    def last_resample_ms(self):
        a, b = C.c_float(), C.c_float()
        self._check(lib().pa_last_resample_ms(self._h, C.byref(a), C.byref(b)), "pa_last_resample_ms")
        return a.value, b.value
