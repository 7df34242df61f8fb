import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: full-size configs (minutes on the GPU box)")


@pytest.fixture(scope="session")
def cfg0():
    """Config 0 (16x16x8 grid, 950 data rows) as numpy CSR + b."""
    import tomogen
    s = tomogen.System(0)
    rp, ci, va = s.csr()
    return dict(sys=s, m=s.dims.m, n=s.dims.n, rp=rp, ci=ci, va=va, b=s.rhs(0), damp=s.damp)


def pytest_sessionfinish(session, exitstatus):
    # stop the background oracle workers of the GPU parity tests (tests/oracle_jobs.py), if any
    mod = sys.modules.get("oracle_jobs")
    if mod is not None:
        mod.shutdown()
