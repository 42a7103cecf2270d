import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size parity case (minutes of oracle time)")


def rel_l2(a, b):
    """||a - b||_2 / ||b||_2 in double, b the reference."""
    import numpy as np
    a = np.asarray(a)
    b = np.asarray(b)
    ad = a.astype(np.complex128 if np.iscomplexobj(a) or np.iscomplexobj(b) else np.float64)
    bd = b.astype(ad.dtype)
    return float(np.linalg.norm((ad - bd).ravel()) / np.linalg.norm(bd.ravel()))


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle
