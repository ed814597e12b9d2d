"""paper_1703_03676_b200 -- population annealing hot path for the 2D Ising model on NVIDIA B200.

`from paper_1703_03676_b200 import pa` gives the ctypes binding of the C-ABI library declared in
include/pa.h (same names: pa_create, pa_sweep, pa_energies, pa_resample, pa_adapt_dbeta,
pa_observables, pa_destroy, ...).  Importing the package itself loads nothing.
"""
__all__ = ["workloads"]
