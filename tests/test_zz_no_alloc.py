"""pa_weighted_average_static: the allocation-free variant of the weighted average over runs (Eq. 6-7).

Why it exists: some users of this library cannot let it call cudaMalloc -- they have already given every byte of the GPU to
their populations (or to a framework's memory pool), or they have other populations sweeping on other streams that a
cudaMalloc / cudaFree pair would bring to a halt, or they call from a place where a blocking driver call is forbidden.  For
them the weights omega_m live in a fixed 32 KiB array inside the library (at most PA_WAVG_STATIC_MAX_RUNS = 4096 runs) and the
call allocates nothing.  What is checked here is that this variant gives what pa_weighted_average (the allocating path) gives, on
calls made one after the other -- the second with fewer runs than the first, so that the array still holds the first call's
weights beyond the part the second one rewrites -- and that sizes beyond the array are refused instead of overrunning it.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure and a failure here must not hide the
parity tests.  It has to pass on its own in a fresh process (where its first call also looks up the array's device address) and
after all the other tests."""
import ctypes as C

import numpy as np
import pytest

from paper_1703_03676_b200 import pa

REL = 1e-9          # the tolerance of the fp64 observables in tests/test_parity_gpu.py


def test_static_limit_is_refused_before_any_cuda_call():
    """More runs than the array holds: a clear error code and text, nothing launched (needs no GPU)."""
    assert pa.lib().pa_weighted_average_static_max_runs() == pa.PA_WAVG_STATIC_MAX_RUNS == 4096
    fake = C.c_void_p(256)                                   # never dereferenced: the size check comes first
    rc = pa.lib().pa_weighted_average_static(pa.PA_WAVG_STATIC_MAX_RUNS + 1, fake, fake, 1, fake, None)
    assert rc == pa.PA_ERR_STATIC_LIMIT
    assert "PA_WAVG_STATIC_MAX_RUNS" in pa.strerror(rc)
    assert pa.lib().pa_weighted_average_static(0, fake, fake, 1, fake, None) == pa.PA_ERR_INVALID_ARG
    assert pa.lib().pa_weighted_average_static(3, None, fake, 1, fake, None) == pa.PA_ERR_INVALID_ARG


def _cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _runs(rng, M, nobs):
    """lnZ of M runs spread over a few units (so that the weights span orders of magnitude) and their observables."""
    return rng.normal(1234.5, 2.0, M), rng.normal(0.0, 1.0, (M, nobs))


@pytest.mark.gpu
def test_static_variant_matches_the_allocating_path_on_consecutive_calls():
    torch = _cuda()
    rng = np.random.default_rng(20261106)
    # 300 runs (more than one pass of the 256 threads), then 7 (stale weights of the first call stay behind them),
    # then the full 4096 the array can hold, then 1 run (weight exactly 1).
    for M, nobs in ((300, 5), (7, 3), (pa.PA_WAVG_STATIC_MAX_RUNS, 4), (1, 2)):
        lnZ, A = _runs(rng, M, nobs)
        want, _ = pa.pa_weighted_average(lnZ, A)                          # the existing path: host pointers, cudaMalloc inside
        d_lnZ, d_A = torch.from_numpy(lnZ).cuda(), torch.from_numpy(A).cuda()
        d_out = torch.full((nobs,), float("nan"), dtype=torch.float64, device="cuda")
        pa.pa_weighted_average_static(d_lnZ, d_A, d_out)                   # asynchronous, on torch's current stream
        torch.cuda.current_stream().synchronize()
        got = d_out.cpu().numpy()
        assert np.allclose(got, want, rtol=REL, atol=0), (M, nobs, got, want)
        if M == 1:
            assert np.array_equal(got, A[0])


@pytest.mark.gpu
def test_static_variant_on_a_side_stream_and_same_input_twice():
    """The same inputs twice in a row on a stream of the caller's give the same bytes; the call does not need the default stream."""
    torch = _cuda()
    rng = np.random.default_rng(7)
    lnZ, A = _runs(rng, 50, 6)
    want, _ = pa.pa_weighted_average(lnZ, A)
    d_lnZ, d_A = torch.from_numpy(lnZ).cuda(), torch.from_numpy(A).cuda()
    outs = [torch.zeros(6, dtype=torch.float64, device="cuda") for _ in range(2)]
    side = torch.cuda.Stream()
    torch.cuda.synchronize()                                               # the inputs are ready before the side stream reads them
    for o in outs:
        pa.pa_weighted_average_static(d_lnZ, d_A, o, cuda_stream=side.cuda_stream)   # same stream: ordered, no race on the array
    side.synchronize()
    a, b = outs[0].cpu().numpy(), outs[1].cpu().numpy()
    assert np.array_equal(a, b)
    assert np.allclose(a, want, rtol=REL, atol=0)


@pytest.mark.gpu
def test_static_variant_refuses_what_it_cannot_do():
    torch = _cuda()
    M = pa.PA_WAVG_STATIC_MAX_RUNS + 1
    d_lnZ = torch.zeros(M, dtype=torch.float64, device="cuda")
    d_A = torch.zeros((M, 1), dtype=torch.float64, device="cuda")
    d_out = torch.full((1,), 5.0, dtype=torch.float64, device="cuda")
    with pytest.raises(pa.PaError) as e:
        pa.pa_weighted_average_static(d_lnZ, d_A, d_out)
    assert e.value.code == pa.PA_ERR_STATIC_LIMIT
    torch.cuda.synchronize()
    assert d_out.item() == 5.0                                             # nothing was launched
    host = np.zeros(4)                                                     # a host pointer where a device pointer is required
    rc = pa.lib().pa_weighted_average_static(4, C.c_void_p(host.ctypes.data), C.c_void_p(d_A.data_ptr()), 1,
                                             C.c_void_p(d_out.data_ptr()), None)
    assert rc == pa.PA_ERR_INVALID_ARG
