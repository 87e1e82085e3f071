import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run with -m gpu through the C-ABI library)")


def relerr(a, b):
    """normwise relative errors (2-norm, inf-norm) of a against reference b (SURVEY 8(c) reading 14)."""
    import numpy as np
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    d = a - b
    n2 = np.linalg.norm(b)
    ni = np.abs(b).max() if b.size else 0.0
    e2 = np.linalg.norm(d) / n2 if n2 > 0 else np.linalg.norm(d)
    ei = np.abs(d).max() / ni if ni > 0 else (np.abs(d).max() if d.size else 0.0)
    return float(e2), float(ei)


@pytest.fixture(scope="session")
def rel():
    return relerr
