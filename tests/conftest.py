import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def smo():
    """The CPU oracle (test infrastructure)."""
    from oracle import smo as _smo
    _smo.lib()
    return _smo


@pytest.fixture(scope="session")
def oracle_force(smo):
    def ff(pot, pts):
        return smo.eval_force(pot, pts, 0.0, want_phi=False)
    return ff
