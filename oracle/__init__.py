"""float64 CPU oracle for the TINA FIR / DFT / PFB path -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this package.  It shares no code with the
CUDA path (``paper_2408_16551_b200``) and never imports it.

The arithmetic lives in ``tina_oracle.c`` (plain loops, double precision, each
function citing the passage of PAPER.md it restates).  This module only builds
that file with gcc and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tina_oracle.c")
_LIB = os.path.join(_HERE, "libtina_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile tina_oracle.c -> libtina_oracle.so (gcc -O2 -fopenmp)."""
    with _lock:
        if (not force and os.path.exists(_LIB)
                and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
            return _LIB
        tmp = _LIB + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O2", "-fopenmp", "-fno-fast-math", "-shared", "-fPIC",
               "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
        return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = ctypes.CDLL(_LIB)
    ll, vp, ci = ctypes.c_longlong, ctypes.c_void_p, ctypes.c_int
    lib.oracle_fir.argtypes = [vp, vp, vp, ll, ll, ll]
    lib.oracle_fir.restype = ci
    lib.oracle_fir_multi.argtypes = [vp, vp, vp, ll, ll, ll]
    lib.oracle_fir_multi.restype = ci
    lib.oracle_unfold.argtypes = [vp, vp, ll, ll]
    lib.oracle_unfold.restype = ci
    lib.oracle_dft.argtypes = [vp, vp, ll, ll, ci]
    lib.oracle_dft.restype = ci
    lib.oracle_dft_f64.argtypes = [vp, vp, ll, ll, ci]
    lib.oracle_dft_f64.restype = ci
    lib.oracle_pfb_num_frames.argtypes = [ll, ll, ll]
    lib.oracle_pfb_num_frames.restype = ll
    lib.oracle_pfb.argtypes = [vp, ll, ll, ll, vp, ci, vp, ll, vp, vp]
    lib.oracle_pfb.restype = ci
    lib.oracle_num_threads.restype = ci
    for name in ("oracle_mul", "oracle_add"):
        getattr(lib, name).argtypes = [vp, vp, vp, ll]
        getattr(lib, name).restype = ci
    lib.oracle_sum.argtypes = [vp, vp, ll, ll]
    lib.oracle_sum.restype = ci
    lib.oracle_matmul.argtypes = [vp, vp, vp, ll, ll, ll]
    lib.oracle_matmul.restype = ci
    lib.oracle_set_num_threads.argtypes = [ci]
    _lib = lib
    return lib


def _ptr(a):
    return ctypes.c_void_p(a.ctypes.data)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def fir(x, taps) -> np.ndarray:
    """Eq. (15), valid mode.  x: [C, L] (or [L]) float32, taps: [K] float32 -> float64 [C, L-K+1]."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    one_d = x.ndim == 1
    if one_d:
        x = x[None, :]
    taps = np.ascontiguousarray(taps, dtype=np.float32)
    C, L = x.shape
    K = taps.shape[0]
    y = np.empty((C, L - K + 1), dtype=np.float64)
    rc = _load().oracle_fir(_ptr(x), _ptr(taps), _ptr(y), C, L, K)
    if rc:
        raise ValueError(f"oracle_fir rc={rc}")
    return y[0] if one_d else y


def fir_multi(x, taps) -> np.ndarray:
    """Eq. (15) with per-channel taps ("multiple FIR filters").
    x: [C, L] float32, taps: [C, K] float32 -> float64 [C, L-K+1]."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    taps = np.ascontiguousarray(taps, dtype=np.float32)
    if x.ndim != 2 or taps.ndim != 2 or taps.shape[0] != x.shape[0]:
        raise ValueError("need x [C, L] and taps [C, K]")
    C, L = x.shape
    K = taps.shape[1]
    y = np.empty((C, L - K + 1), dtype=np.float64)
    rc = _load().oracle_fir_multi(_ptr(x), _ptr(taps), _ptr(y), C, L, K)
    if rc:
        raise ValueError(f"oracle_fir_multi rc={rc}")
    return y


def unfold(x, J: int) -> np.ndarray:
    """Eq. (17): Y(i,j) = X(i+j), shape (I-J+1, J)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    I = x.shape[0]
    y = np.empty((I - J + 1, J), dtype=np.float64)
    rc = _load().oracle_unfold(_ptr(x), _ptr(y), I, J)
    if rc:
        raise ValueError(f"oracle_unfold rc={rc}")
    return y


def _binary(name, a, b):
    a = np.ascontiguousarray(a, dtype=np.float32)
    b = np.ascontiguousarray(b, dtype=np.float32)
    if a.shape != b.shape:
        raise ValueError("shape mismatch")
    o = np.empty(a.shape, dtype=np.float64)
    rc = getattr(_load(), name)(_ptr(a), _ptr(b), _ptr(o), a.size)
    if rc:
        raise ValueError(f"{name} rc={rc}")
    return o


def mul(a, b) -> np.ndarray:
    """Eq. (6): elementwise product of two float32 arrays -> float64."""
    return _binary("oracle_mul", a, b)


def add(a, b) -> np.ndarray:
    """Eq. (10): elementwise sum of two float32 arrays -> float64."""
    return _binary("oracle_add", a, b)


def summation(x) -> np.ndarray:
    """Eq. (11): sum over the last axis.  x: [rows, n] (or [n]) float32 -> float64 [rows] (or scalar array)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    one_d = x.ndim == 1
    if one_d:
        x = x[None, :]
    rows, n = x.shape
    o = np.empty(rows, dtype=np.float64)
    rc = _load().oracle_sum(_ptr(x), _ptr(o), rows, n)
    if rc:
        raise ValueError(f"oracle_sum rc={rc}")
    return o[0] if one_d else o


def matmul(x, y) -> np.ndarray:
    """Eq. (7): Z = X Y.  x: [M, L], y: [L, N] float32 -> float64 [M, N]."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    M, L = x.shape
    L2, N = y.shape
    if L != L2:
        raise ValueError("inner dimensions differ")
    z = np.empty((M, N), dtype=np.float64)
    rc = _load().oracle_matmul(_ptr(x), _ptr(y), _ptr(z), M, L, N)
    if rc:
        raise ValueError(f"oracle_matmul rc={rc}")
    return z


def dft(x, inverse: bool = False) -> np.ndarray:
    """Eq. (12)/(14).  x: [B, N] (or [N]) complex64 or complex128 -> complex128."""
    x = np.asarray(x)
    one_d = x.ndim == 1
    if one_d:
        x = x[None, :]
    B, N = x.shape
    z = np.empty((B, N), dtype=np.complex128)
    if x.dtype == np.complex128:
        x = np.ascontiguousarray(x)
        rc = _load().oracle_dft_f64(_ptr(x), _ptr(z), B, N, int(bool(inverse)))
    else:
        x = np.ascontiguousarray(x, dtype=np.complex64)
        rc = _load().oracle_dft(_ptr(x), _ptr(z), B, N, int(bool(inverse)))
    if rc:
        raise ValueError(f"oracle_dft rc={rc}")
    return z[0] if one_d else z


def pfb_num_frames(n_samples: int, P: int, M: int) -> int:
    return int(_load().oracle_pfb_num_frames(n_samples, P, M))


def pfb(x, P: int, M: int, window, frames=None, return_subfiltered: bool = False):
    """Eq. (20) + DFT.  x: 1-D complex64 (complex kind) or float32 (real kind).

    Returns X [n_sel, P] (complex kind) or [n_sel, P/2+1] (real kind), complex128;
    with return_subfiltered also y [n_sel, P] (complex128 / float64).
    ``frames``: optional 1-D int array of frame indices (default: all frames).
    """
    x = np.asarray(x)
    is_real = not np.iscomplexobj(x)
    x = np.ascontiguousarray(x, dtype=np.float32 if is_real else np.complex64)
    w = np.ascontiguousarray(window, dtype=np.float32)
    n = x.shape[0]
    if w.shape[0] != P * M:
        raise ValueError("window must have P*M entries")
    F = pfb_num_frames(n, P, M)
    if F < 1:
        raise ValueError("too few samples")
    if frames is None:
        fr, n_sel, frp = None, F, ctypes.c_void_p(0)
    else:
        fr = np.ascontiguousarray(frames, dtype=np.int64)
        n_sel, frp = fr.shape[0], _ptr(fr)
    NK = P // 2 + 1 if is_real else P
    X = np.empty((n_sel, NK), dtype=np.complex128)
    if return_subfiltered:
        y = np.empty((n_sel, P), dtype=np.float64 if is_real else np.complex128)
        yp = _ptr(y)
    else:
        y, yp = None, ctypes.c_void_p(0)
    rc = _load().oracle_pfb(_ptr(x), n, P, M, _ptr(w), int(is_real), frp, n_sel, yp, _ptr(X))
    if rc:
        raise ValueError(f"oracle_pfb rc={rc}")
    return (X, y) if return_subfiltered else X
