"""Seeded synthetic workloads: the five configurations of BASELINE.json and their beta schedules.

This module serves BOTH the CUDA path's harness and the CPU oracle's tests, and therefore holds
none of the method's arithmetic: only shapes (L, R), seeds, sweep counts and the list of inverse
temperatures, which is handed to both sides as data ("input recipe").
It imports neither the binding nor the oracle.

The paper measures on no external dataset: its workloads are populations of random-start Ising
replicas (Tables 2-3: L = 16..256, R = 2 000..100 000, theta = 1..500).  The spins
themselves are generated inside each implementation from the seed (INIT stream, O1).
"""
from dataclasses import dataclass
from typing import List, Optional, Tuple


@dataclass(frozen=True)
class Workload:
    name: str
    L: int                 # lattice edge, periodic L x L
    R: int                 # target population size
    seed: int              # Philox key
    beta0: float
    beta_f: float
    n_steps: Optional[int]          # equal steps; None = adaptive
    theta: int                      # Metropolis sweeps per temperature (L61)
    target_overlap: Optional[float] = None   # alpha* of Eq. 8 (L115) when adaptive
    multi_histogram: bool = False            # Eq. 9 accumulation at every temperature
    dims: Optional[Tuple[int, int, int]] = None   # (Lx, Ly, Lz) of a simple-cubic box; None = L x L square lattice

    @property
    def N(self) -> int:
        return self.L * self.L if self.dims is None else self.dims[0] * self.dims[1] * self.dims[2]

    @property
    def groups(self) -> int:
        return (self.R + 31) // 32

    def betas(self) -> List[float]:
        """beta_i = beta0 + (beta_f - beta0) * i / n, i = 0..n (O10 reading)."""
        assert self.n_steps is not None, "adaptive workload: the schedule is produced by pa_adapt_dbeta"
        n = self.n_steps
        return [self.beta0 + (self.beta_f - self.beta0) * float(i) / float(n) for i in range(n + 1)]


CONFIGS = {
    1: Workload("cfg1_L16_R1000", 16, 1000, 1, 0.0, 1.0, 100, 10),
    2: Workload("cfg2_L64_R20000", 64, 20000, 2, 0.0, 1.0, 200, 10),
    3: Workload("cfg3_L64_R131072", 64, 131072, 3, 0.0, 1.0, 200, 10),
    4: Workload("cfg4_L128_R100000_adaptive", 128, 100000, 4, 0.0, 1.0, None, 10,
                target_overlap=0.85, multi_histogram=True),
    5: Workload("cfg5_L256_R1000000", 256, 1000000, 5, 0.0, 0.5, 500, 10),
    # not in BASELINE.json: SURVEY 8(f) row 4, the second workload on another lattice ("models on different lattices in
    # various dimensions", L43 "3D Ising systems"): a 32^3 simple-cubic lattice, R = 100 000, beta 0 -> 0.3 (past beta_c = 0.2217)
    6: Workload("cube_L32_R100000", 32, 100000, 6, 0.0, 0.3, 150, 10, dims=(32, 32, 32)),
}


def table3_workload(theta: int, R: int = 50000) -> Workload:
    """The shape of the paper's theta scan (Table 3 / Table 4 / Table 5: L = 128, R = 50 000,
    theta = 1 .. 500 on a Tesla K80).  The paper does not restate the temperature step for these tables; Table 1's
    (L189: dbeta = 0.02, i.e. 50 equal steps from 0 to 1) is used -- t_SF is normalised per spin flip, so the number of
    temperatures only sets how often the resampling cost is paid per theta sweeps, which is once in either case."""
    return Workload(f"table3_L128_R{R}_theta{theta}", 128, R, 7, 0.0, 1.0, 50, theta)


def random_couplings(L: int, seed: int):
    """A seeded bimodal sample for the second workload (O15): independent J = +-1 with probability 1/2 on
    every bond of the L x L torus (the 2D Edwards-Anderson +-J spin glass).  Returns (Jx, Jy), int8 [L*L] each, site = y*L + x."""
    import numpy as np
    rng = np.random.default_rng(seed)
    Jx = (rng.integers(0, 2, L * L) * 2 - 1).astype(np.int8)
    Jy = (rng.integers(0, 2, L * L) * 2 - 1).astype(np.int8)
    return Jx, Jy
