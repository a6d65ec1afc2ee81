import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    import oracle as _oracle
    _oracle.build()
    return _oracle


def rel_l2_rows(got, ref):
    """max over rows of ||got_r - ref_r||_2 / ||ref_r||_2 (the contractual per-frame metric, R14)."""
    import numpy as np
    got = np.asarray(got).reshape(ref.shape[0], -1).astype(np.complex128)
    ref2 = np.asarray(ref).reshape(ref.shape[0], -1).astype(np.complex128)
    num = np.linalg.norm(got - ref2, axis=1)
    den = np.linalg.norm(ref2, axis=1)
    den = np.where(den == 0, 1.0, den)
    return float((num / den).max())
