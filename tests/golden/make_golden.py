"""Writes the stored expected values under tests/golden/.  Calls only oracle/ (never the CUDA path).

    python tests/golden/make_golden.py

ising_4x4_dos.txt : density of states g(E) of the 4x4 periodic Ising model by enumeration of all
                    2^16 states (oracle/exact_ising.py).  The same numbers are the textbook
                    result for this lattice (e.g. P. D. Beale, Phys. Rev. Lett. 76 (1996) 78,
                    who expands Kaufman's solution, PAPER.md ref. [28] context L361);
                    sum = 65536, symmetric under E -> -E, no states at E = +-28.
kaufman_L16.txt   : exact ln Z, e, C of the 16x16 torus at five inverse temperatures from
                    Kaufman's formula (oracle/exact_ising.py: kaufman), 60-digit arithmetic.
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import exact_ising as ex  # noqa: E402

with open(os.path.join(HERE, "ising_4x4_dos.txt"), "w") as f:
    f.write("# E  g(E)   4x4 periodic Ising model, all 65536 states (see make_golden.py)\n")
    for E, g in sorted(ex.density_of_states(4).items()):
        f.write(f"{E} {g}\n")

with open(os.path.join(HERE, "kaufman_L16.txt"), "w") as f:
    f.write("# beta  lnZ  e  C    16x16 periodic Ising model, Kaufman's formula (see make_golden.py)\n")
    for beta in (0.1, 0.3, 0.44, 0.6, 1.0):
        k = ex.kaufman(beta, 16)
        f.write(f"{beta!r} {k['lnZ']!r} {k['e']!r} {k['C']!r}\n")
