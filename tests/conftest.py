import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: takes more than a few seconds on CPU")


def rel_err(a, b, denom=None):
    """||a-b||_2 / ||b||_2 on svec vectors (= Frobenius on matrices).
    If ||b|| = 0 the caller passes the input norm as `denom`."""
    import numpy as np
    d = np.linalg.norm(b) if denom is None else denom
    if d == 0.0:
        d = 1.0
    return float(np.linalg.norm(a - b) / d)


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.build()
    return oracle
