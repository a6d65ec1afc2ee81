"""NumPy-style vectorised CPU PFB -- TEST / BASELINE INFRASTRUCTURE (never on the product path).

The stand-in for the paper's "naive implementation written in NumPy (on CPU)"
(PAPER.md:235): reshape to [blocks, P], M shifted slice multiply-accumulates with
the window rows (Eq. (20), reading R6), then numpy.fft along the
channel axis ("either a Discrete or Fast Fourier Transform").
complex64 / float32 arithmetic.  It is a *reported* CPU baseline in bench.py and a
second, independent check of the branch-order readings R4-R6 against the float64
oracle (tests/test_numpy_baseline.py).
"""
from __future__ import annotations

import numpy as np


def pfb_subfilter(x: np.ndarray, P: int, M: int, window: np.ndarray) -> np.ndarray:
    nb = x.shape[0] // P
    F = nb - M + 1
    xb = x[: nb * P].reshape(nb, P)
    w = np.asarray(window, dtype=np.float32).reshape(M, P)
    y = np.zeros((F, P), dtype=xb.dtype)
    for m in range(M):
        # tap row m multiplies the block m steps in the past: block index f + M-1 - m
        y += w[m][None, :] * xb[M - 1 - m: M - 1 - m + F]
    return y


def pfb(x: np.ndarray, P: int, M: int, window: np.ndarray) -> np.ndarray:
    y = pfb_subfilter(x, P, M, window)
    if np.iscomplexobj(y):
        return np.fft.fft(y, axis=1).astype(np.complex64)
    return np.fft.rfft(y, axis=1).astype(np.complex64)
