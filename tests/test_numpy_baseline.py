"""The NumPy-style CPU baseline (oracle/numpy_pfb.py) agrees with the float64 oracle (CPU only)."""
import numpy as np
import pytest

import tina_inputs as ti
from conftest import rel_l2_rows


@pytest.mark.parametrize("real", [False, True])
def test_numpy_pfb_matches_oracle(oracle, real):
    from oracle import numpy_pfb
    P, M, F = 32, 4, 50
    rng = np.random.default_rng(7)
    c = ti.pfb_case(P, M, F, real=real, seed=8, window=ti.random_taps(rng, P * M))
    ref, yref = oracle.pfb(c.x[0], P, M, c.window, return_subfiltered=True)
    assert rel_l2_rows(numpy_pfb.pfb_subfilter(c.x[0], P, M, c.window), yref) < 1e-5
    assert rel_l2_rows(numpy_pfb.pfb(c.x[0], P, M, c.window), ref) < 1e-5


def test_config1_numpy_vs_oracle(oracle):
    from oracle import numpy_pfb
    c = ti.config1()
    assert c.x.shape == (1, 65584) and c.n_frames == 4096
    ref = oracle.pfb(c.x[0], c.P, c.M, c.window)
    assert ref.shape == (4096, 16)
    assert rel_l2_rows(numpy_pfb.pfb(c.x[0], c.P, c.M, c.window), ref) < 1e-5
