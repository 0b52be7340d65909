import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def orc():
    """The CPU oracle (builds oracle/liboracle.so with gcc on first use)."""
    import oracle
    oracle.build()
    return oracle


def rel_err(a, b):
    """max|a-b| / max|b| -- the parity metric of BASELINE.json:north_star."""
    import numpy as np
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    m = float(np.max(np.abs(b))) if b.size else 0.0
    if m == 0.0:
        return float(np.max(np.abs(a - b))) if b.size else 0.0
    return float(np.max(np.abs(a - b)) / m)
