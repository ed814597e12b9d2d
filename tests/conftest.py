import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def cfg1_oracle_runs():
    """configs[0] of BASELINE.json (L=16, R=1000, 100 equal steps to beta=1, theta=10) on the CPU oracle, seeds 1..16, one Philox
    number per spin, Eq. 9 sums accumulated: computed once per session and shared by the Kaufman pins of the observables,
    of the reweighting, and by the variance-ratio pin of the LCG-assisted stream.  Returns [(oracle, observables per beta)]."""
    from oracle import pa_oracle as po
    import pa_driver
    betas = [i / 100 for i in range(101)]
    out = []
    for seed in range(1, 17):
        o = po.Oracle(16, 1000, seed)
        out.append((o, pa_driver.run_fixed(o, betas, 10, hist=True)))
    return betas, out
