"""The exact references used as pins are themselves cross-checked here: Kaufman's closed form
(typed from the textbook formula) against brute-force enumeration at L = 4, against known
limits, and against the stored golden values."""
import math
import os

import numpy as np
import pytest

from oracle import exact_ising as ex

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_dos_4x4_golden_and_symmetries():
    g = ex.density_of_states(4)
    gold = {int(a): int(b) for a, b in (l.split() for l in open(os.path.join(GOLD, "ising_4x4_dos.txt")) if l[0] != "#")}
    assert g == gold
    assert sum(g.values()) == 2**16
    assert all(g[E] == g[-E] for E in g)
    assert g[-32] == 2 and -28 not in g and g[-24] == 32        # ground states; one flipped spin: 2*16
    assert g[-20] == 64                                          # two adjacent flipped spins: 2*32 bonds


@pytest.mark.parametrize("beta", [0.05, 0.2, 0.4406868, 0.8, 1.5])
def test_kaufman_equals_enumeration_L4(beta):
    a, k = ex.exact_small(beta, 4), ex.kaufman(beta, 4)
    assert k["lnZ"] == pytest.approx(a["lnZ"], rel=1e-13)
    assert k["e"] == pytest.approx(a["e"], rel=1e-11)
    assert k["C"] == pytest.approx(a["C"], rel=1e-8)
    assert k["S_per_N"] == pytest.approx(a["S_per_N"], rel=1e-10)


def test_kaufman_limits_and_golden():
    for L in (16, 64, 256):
        N = L * L
        assert float(ex.kaufman_lnZ(1e-9, L)) == pytest.approx(N * math.log(2), rel=1e-12)   # Z(0) = 2^N (L93)
        k = ex.kaufman(3.0, L)
        assert k["e"] == pytest.approx(-2.0, abs=1e-3)                                          # ground state
        assert k["lnZ"] == pytest.approx(2 * N * 3.0 + math.log(2), rel=1e-6)
    # thermodynamic limit at beta_c: e = -sqrt(2) (Onsager); finite L approaches it from below
    e64, e256 = ex.kaufman(ex.BETA_C, 64)["e"], ex.kaufman(ex.BETA_C, 256)["e"]
    assert e64 < e256 < -math.sqrt(2) and abs(e256 + math.sqrt(2)) < 0.01
    for line in open(os.path.join(GOLD, "kaufman_L16.txt")):
        if line[0] == "#":
            continue
        beta, lnZ, e, C = map(float, line.split())
        k = ex.kaufman(beta, 16)
        assert (k["lnZ"], k["e"], k["C"]) == pytest.approx((lnZ, e, C), rel=1e-12)
