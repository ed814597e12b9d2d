"""The C-ABI library builds for sm_100a on a CPU-only box, loads, and exports every symbol that
include/pa.h declares; host-only entry points behave; there is no CPU fallback (-m "not gpu")."""
import ctypes as C
import os
import re
import subprocess

import pytest

from paper_1703_03676_b200 import build as pa_build
from paper_1703_03676_b200 import pa

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    return pa_build.build()


def test_library_exports_every_declared_symbol(libpath):
    declared = pa.declared_symbols()
    assert len(declared) >= 30 and "pa_create" in declared and "pa_sweep" in declared and "pa_resample" in declared
    out = subprocess.run(["nm", "-D", "--defined-only", libpath], check=True, capture_output=True, text=True).stdout
    exported = {line.split()[-1] for line in out.splitlines() if " T " in line}
    missing = [s for s in declared if s not in exported]
    assert not missing, missing
    L = pa.lib()
    for s in declared:
        assert hasattr(L, s)


def test_library_contains_sm100a_code(libpath):
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_host_only_entry_points():
    assert pa.pa_capacity(1000) == 32 * ((1000 + 1024 + 31) // 32)
    assert pa.pa_capacity(1000000) == 32 * ((1000000 + 8000 + 31) // 32)
    assert pa.pa_workspace_bytes(256, 1000000) > 2 * 31250 * 65536 * 4          # two packed buffers at cfg 5
    assert pa.pa_workspace_bytes(256, 1000000) < 20 * 2**30
    n = C.c_size_t()
    assert pa.lib().pa_workspace_bytes(15, 100, C.byref(n)) == pa.PA_ERR_INVALID_ARG   # odd L
    assert pa.lib().pa_workspace_bytes(2, 100, C.byref(n)) == pa.PA_ERR_INVALID_ARG
    assert pa.lib().pa_workspace_bytes(16, 0, C.byref(n)) == pa.PA_ERR_INVALID_ARG
    assert pa.strerror(pa.PA_ERR_CAPACITY).startswith("resampled population")
    assert pa.lib().pa_version().decode().startswith("pa-b200")


@pytest.fixture(scope="module")
def c_client(libpath, tmp_path_factory):
    """include/pa.h compiles as strict C99 and a C program links against the library."""
    exe = str(tmp_path_factory.mktemp("abi") / "abi_c_client")
    pkg = os.path.dirname(libpath)
    subprocess.run(["gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                    os.path.join(ROOT, "tests", "helpers", "abi_c_client.c"), "-o", exe,
                    "-L", pkg, "-lpa_b200", "-Wl,-rpath," + pkg], check=True)
    return exe


def test_c_client_links_and_reports_no_device(c_client):
    import torch
    r = subprocess.run([c_client], capture_output=True, text=True)
    if torch.cuda.is_available():
        assert r.returncode == 0, r.stdout + r.stderr
    else:
        assert r.returncode == 3 and "no device" in r.stdout          # PA_ERR_CUDA from pa_create: no CPU fallback


@pytest.mark.gpu
def test_c_client_runs_the_paper_loop(c_client):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    r = subprocess.run([c_client, "32", "3000"], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    lines = r.stdout.strip().splitlines()
    assert len(lines) >= 4 and lines[-2].startswith("reweighted to beta=0.25")
    assert lines[-1].startswith("host step to beta=0.55") and -2.0 < float(lines[-1].split("e=")[1].split()[0]) < -1.0   # pa_step_host, pageable buffers
    last = lines[-3].split()
    betas = [float(l.split()[0]) for l in lines[:-2]]
    assert all(b > a for a, b in zip(betas, betas[1:])) and 0.0 < betas[-1] <= 0.5    # the adaptive schedule moves forward
    assert -2.0 < float(last[1]) < 0.0 and abs(float(last[1]) + 2.0 * betas[-1]) < 0.1   # e ~ -2 beta at high temperature


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present: the fallback check is for CPU-only boxes")
    h = C.c_void_p()
    assert pa.lib().pa_create(16, 64, 1, C.byref(h)) == pa.PA_ERR_CUDA
    with pytest.raises(pa.PaError):
        pa.Population(16, 64, 1)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1703_03676_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+\.*oracle", text, flags=re.M), f
                assert not re.search(r"#include\s*[<\"][^>\"]*oracle", text), f
