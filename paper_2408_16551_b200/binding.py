"""ctypes binding of libtina.so -- argument marshalling only; every step runs in the CUDA kernels.

Functions mirror include/tina.h: fir <-> tina_fir, dft <-> tina_dft, pfb <-> tina_pfb_batched,
pfb_fir <-> tina_pfb_fir_batched, pfb_host <-> tina_pfb_batched_host.
The library is loaded lazily; a missing or unloadable libtina.so raises (no fallback of any kind).
"""
from __future__ import annotations

import ctypes
import os

COMPLEX, REAL = 0, 1
PREC_FP32, PREC_BF16, PREC_FP16 = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtina.so")
_lib = None

EXPORTS = ["tina_fir", "tina_fir_multi", "tina_unfold", "tina_dft", "tina_pfb", "tina_pfb_batched", "tina_pfb_fir_batched", "tina_pfb_fft_batched",
           "tina_pfb_batched_host", "tina_pfb_num_frames", "tina_status_string", "tina_last_error",
           "tina_clear_plan_cache", "tina_version", "tina_launch_count", "tina_last_path", "tina_reload_options", "tina_build_is_dev", "tina_probe_peak", "tina_last_kernel", "tina_last_issued_ratio",
           "tina_mul", "tina_add", "tina_sum", "tina_sum_static", "tina_matmul"]


class TinaError(RuntimeError):
    def __init__(self, status: int, name: str, detail: str):
        super().__init__(f"{name} ({status}): {detail}")
        self.status, self.name, self.detail = status, name, detail


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2408_16551_b200.build` "
                          "(or __graft_entry__.build()); there is no fallback path")
    L = ctypes.CDLL(_LIB_PATH)
    ll, vp, ci = ctypes.c_longlong, ctypes.c_void_p, ctypes.c_int
    L.tina_fir.argtypes = [vp, vp, vp, ci, ll, ci, vp]
    L.tina_fir_multi.argtypes = [vp, vp, vp, ci, ll, ci, vp]
    L.tina_fir_multi.restype = ci
    L.tina_unfold.argtypes = [vp, vp, ll, ci, vp]
    L.tina_dft.argtypes = [vp, vp, ll, ci, ci, ci, vp]
    L.tina_pfb.argtypes = [vp, ll, ci, ci, vp, ci, ci, vp, vp]
    L.tina_pfb_batched.argtypes = [vp, ci, ll, ci, ci, vp, ci, ci, vp, vp]
    L.tina_pfb_fir_batched.argtypes = [vp, ci, ll, ci, ci, vp, ci, vp, vp]
    L.tina_pfb_fft_batched.argtypes = [vp, ci, ll, ci, ci, vp, ci, vp, vp]
    L.tina_pfb_batched_host.argtypes = [vp, ci, ll, ci, ci, vp, ci, ci, vp, vp]
    L.tina_mul.argtypes = [vp, vp, vp, ll, vp]
    L.tina_add.argtypes = [vp, vp, vp, ll, vp]
    L.tina_sum.argtypes = [vp, ll, ll, vp, vp]
    L.tina_sum_static.argtypes = [vp, ll, ll, vp, vp]
    L.tina_matmul.argtypes = [vp, vp, vp, ll, ll, ll, vp]
    for f in ("tina_mul", "tina_add", "tina_sum", "tina_sum_static", "tina_matmul"):
        getattr(L, f).restype = ci
    for f in ("tina_fir", "tina_unfold", "tina_dft", "tina_pfb", "tina_pfb_batched", "tina_pfb_fir_batched", "tina_pfb_fft_batched",
              "tina_pfb_batched_host", "tina_clear_plan_cache", "tina_version", "tina_last_path", "tina_reload_options",
              "tina_build_is_dev"):
        getattr(L, f).restype = ci
    L.tina_probe_peak.argtypes = [ci, ci, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), vp]
    L.tina_probe_peak.restype = ci
    L.tina_last_kernel.restype = ctypes.c_char_p
    L.tina_last_issued_ratio.restype = ctypes.c_double
    L.tina_pfb_num_frames.argtypes = [ll, ci, ci]
    L.tina_pfb_num_frames.restype = ll
    L.tina_launch_count.restype = ll
    L.tina_status_string.argtypes = [ci]
    L.tina_status_string.restype = ctypes.c_char_p
    L.tina_last_error.restype = ctypes.c_char_p
    _lib = L
    return L


def _check(st: int) -> None:
    if st != 0:
        L = lib()
        raise TinaError(st, L.tina_status_string(st).decode(), L.tina_last_error().decode())


def _stream_ptr(stream, device=None) -> int:
    """Raw CUDA stream handle: `stream` (a torch.cuda.Stream), else torch's current stream on `device` (a torch.device
    of the call's tensors; the current device when None)."""
    import torch
    if stream is None:
        try:        # raw handle of torch's current stream without building a Stream object (a few microseconds per call)
            idx = device.index if (device is not None and device.index is not None) else torch.cuda.current_device()
            return int(torch._C._cuda_getCurrentRawStream(idx))
        except AttributeError:
            stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dev(t, dtype, what):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{what}: expected a CUDA tensor")
    if t.dtype != dtype:
        raise TypeError(f"{what}: expected dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{what}: must be contiguous")
    return t


def _out(out, shape, dtype, device, what="out"):
    """Allocate the result, or check a caller-supplied one: dtype, device, contiguity AND shape
    (a too-small buffer would be overrun by the kernels)."""
    import torch
    shape = tuple(int(v) for v in shape)
    if out is None:
        return torch.empty(shape, dtype=dtype, device=device)
    _dev(out, dtype, what)
    if out.device != device:
        raise ValueError(f"{what}: on {out.device}, inputs on {device}")
    if tuple(out.shape) != shape:
        raise ValueError(f"{what}: expected shape {shape}, got {tuple(out.shape)}")
    return out


def pfb_num_frames(n_samples: int, P: int, M: int) -> int:
    return int(lib().tina_pfb_num_frames(n_samples, P, M))


def launch_count() -> int:
    return int(lib().tina_launch_count())


def last_path() -> int:
    return int(lib().tina_last_path())


def last_kernel() -> str:
    return lib().tina_last_kernel().decode()


def last_issued_ratio() -> float:
    return float(lib().tina_last_issued_ratio())


def clear_plan_cache() -> None:
    _check(lib().tina_clear_plan_cache())


PEAK_FFMA, PEAK_FFMA2, PEAK_TF32, PEAK_BF16 = 0, 1, 2, 3


def probe_peak(which: int, iters: int, stream=None):
    """tina_probe_peak: (TFLOP/s, ms) of a bare FMA / tcgen05.mma loop on the current device."""
    tf, ms = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(lib().tina_probe_peak(which, iters, ctypes.byref(tf), ctypes.byref(ms), _stream_ptr(stream)))
    return tf.value, ms.value


def reload_options() -> None:
    """Re-read the TINA_* variant switches from the environment (they are read once otherwise)."""
    _check(lib().tina_reload_options())


def build_is_dev() -> bool:
    """True if libtina.so was compiled with -DTINA_DEV (work-skipping debug knobs present)."""
    return bool(lib().tina_build_is_dev())


def version() -> int:
    return int(lib().tina_version())


def fir(x, taps, out=None, stream=None):
    """tina_fir: x [C, L] float32 CUDA, taps [M] float32 CUDA -> y [C, L-M+1] float32."""
    import torch
    x = _dev(x, torch.float32, "x")
    taps = _dev(taps, torch.float32, "taps")
    if x.dim() != 2 or taps.dim() != 1:
        raise ValueError("x must be [C, L], taps [M]")
    C, L = x.shape
    M = taps.shape[0]
    out = _out(out, (C, max(L - M + 1, 0)), torch.float32, x.device)
    _check(lib().tina_fir(x.data_ptr(), taps.data_ptr(), out.data_ptr(), C, L, M, _stream_ptr(stream, x.device)))
    return out


def fir_multi(x, taps, out=None, stream=None):
    """tina_fir_multi: x [C, L] float32 CUDA, taps [C, M] float32 CUDA (row c = channel c's taps)
    -> y [C, L-M+1] float32."""
    import torch
    x = _dev(x, torch.float32, "x")
    taps = _dev(taps, torch.float32, "taps")
    if x.dim() != 2 or taps.dim() != 2 or taps.shape[0] != x.shape[0]:
        raise ValueError("x must be [C, L], taps [C, M]")
    C, L = x.shape
    M = taps.shape[1]
    out = _out(out, (C, max(L - M + 1, 0)), torch.float32, x.device)
    _check(lib().tina_fir_multi(x.data_ptr(), taps.data_ptr(), out.data_ptr(), C, L, M, _stream_ptr(stream, x.device)))
    return out


def unfold(x, J: int, out=None, stream=None):
    """tina_unfold: x [I] float32 CUDA -> y [I-J+1, J] float32, Y(i, j) = X(i + j)."""
    import torch
    x = _dev(x, torch.float32, "x")
    if x.dim() != 1:
        raise ValueError("x must be 1-D")
    I = x.shape[0]
    out = _out(out, (max(I - J + 1, 0), J), torch.float32, x.device)
    _check(lib().tina_unfold(x.data_ptr(), out.data_ptr(), I, J, _stream_ptr(stream)))
    return out


def _ew(fn, a, b, out, stream):
    import torch
    a, b = _dev(a, torch.float32, "a"), _dev(b, torch.float32, "b")
    if a.shape != b.shape:
        raise ValueError("a and b must have the same shape")
    out = _out(out, a.shape, torch.float32, a.device)
    _check(fn(a.data_ptr(), b.data_ptr(), out.data_ptr(), a.numel(), _stream_ptr(stream)))
    return out


def mul(a, b, out=None, stream=None):
    """tina_mul, Eq. (6): elementwise product of two float32 CUDA tensors."""
    return _ew(lib().tina_mul, a, b, out, stream)


def add(a, b, out=None, stream=None):
    """tina_add, Eq. (10): elementwise sum of two float32 CUDA tensors."""
    return _ew(lib().tina_add, a, b, out, stream)


def summation(x, out=None, stream=None):
    """tina_sum, Eq. (11): sum over the last axis.  x [rows, n] (or [n]) float32 CUDA -> [rows] (or 0-d)."""
    import torch
    x = _dev(x, torch.float32, "x")
    one_d = x.dim() == 1
    if one_d:
        x = x[None, :]
    if x.dim() != 2:
        raise ValueError("x must be 1-D or 2-D")
    rows, n = x.shape
    out = _out(out, (rows,), torch.float32, x.device)
    _check(lib().tina_sum(x.data_ptr(), rows, n, out.data_ptr(), _stream_ptr(stream)))
    return out[0] if one_d else out


def summation_static(x, out, stream=None):
    """tina_sum_static: tina_sum with its partial sums in a static device array (no device allocation inside the
    call, so `out` [rows] (or 0-d for 1-D x) must be supplied); rows <= 4096; calls that overlap on the GPU race."""
    import torch
    x = _dev(x, torch.float32, "x")
    if x.dim() == 1:
        x = x[None, :]
    if x.dim() != 2:
        raise ValueError("x must be 1-D or 2-D")
    rows, n = x.shape
    if out is None or out.numel() != rows:
        raise ValueError("summation_static needs a preallocated out of rows elements")
    out = _dev(out, torch.float32, "out")
    _check(lib().tina_sum_static(x.data_ptr(), rows, n, out.data_ptr(), _stream_ptr(stream)))
    return out


def matmul(x, y, out=None, stream=None):
    """tina_matmul, Eq. (7): x [M, L] @ y [L, N] -> [M, N], float32 CUDA, row-major."""
    import torch
    x, y = _dev(x, torch.float32, "x"), _dev(y, torch.float32, "y")
    if x.dim() != 2 or y.dim() != 2 or x.shape[1] != y.shape[0]:
        raise ValueError("need x [M, L] and y [L, N]")
    M, L = x.shape
    N = y.shape[1]
    out = _out(out, (M, N), torch.float32, x.device)
    _check(lib().tina_matmul(x.data_ptr(), y.data_ptr(), out.data_ptr(), M, L, N, _stream_ptr(stream)))
    return out


def dft(x, inverse: bool = False, prec: int = PREC_FP32, out=None, stream=None):
    """tina_dft: x [B, N] complex64 CUDA -> [B, N] complex64."""
    import torch
    x = _dev(x, torch.complex64, "x")
    if x.dim() != 2:
        raise ValueError("x must be [B, N]")
    B, N = x.shape
    out = _out(out, x.shape, torch.complex64, x.device)
    _check(lib().tina_dft(x.data_ptr(), out.data_ptr(), B, N, int(bool(inverse)), prec, _stream_ptr(stream, x.device)))
    return out


def _pfb_args(x, P, M, window):
    """Checks of a PFB call's inputs WITHOUT building tensor views (a view costs more than the launch of a small
    problem): returns kind, S, n_samples, F and whether x was one-dimensional."""
    import torch
    nd = x.dim()
    if nd == 1:
        S, n = 1, x.shape[0]
    elif nd == 2:
        S, n = x.shape
    else:
        raise ValueError("x must be [n_samples] or [S, n_samples]")
    if x.dtype == torch.complex64:
        kind = COMPLEX
    elif x.dtype == torch.float32:
        kind = REAL
    else:
        raise TypeError("x must be complex64 (complex kind) or float32 (real kind)")
    if not (x.is_cuda and x.is_contiguous()):
        _dev(x, x.dtype, "x")                                  # raises with the reason
    if not (window.is_cuda and window.dtype == torch.float32 and window.is_contiguous()):
        _dev(window, torch.float32, "window")
    if window.numel() != P * M:
        raise ValueError("window must have P*M entries")
    F = n // P - M + 1 if (P >= 1 and M >= 1) else 0         # tina_pfb_num_frames (include/tina.h)
    return kind, S, n, F, nd == 1


def _pfb_out(out, squeeze, S, F, last, dtype, device):
    """The result buffer of a PFB call: [S, F, last], or [F, last] for a one-dimensional x (a caller-supplied buffer
    of either form is accepted then).  Returns (buffer whose data_ptr is passed, tensor handed back to the caller)."""
    import torch
    F = max(F, 0)
    if out is None:
        out = torch.empty((F, last) if squeeze else (S, F, last), dtype=dtype, device=device)
        return out, out
    if squeeze and out.dim() == 3:
        _out(out, (1, F, last), dtype, device)
        return out, out[0]
    shape = (F, last) if squeeze else (S, F, last)
    if not (out.is_cuda and out.dtype == dtype and out.shape == shape and out.device == device and out.is_contiguous()):
        _out(out, shape, dtype, device)                        # raises with the reason
    return out, out


def pfb(x, P: int, M: int, window, prec: int = PREC_FP32, out=None, stream=None):
    """tina_pfb_batched: x [S, n_samples] (or [n_samples]) complex64 | float32 CUDA,
    window [P*M] float32 CUDA -> [S, F, P] (complex kind) or [S, F, P/2+1] (real kind) complex64."""
    import torch
    kind, S, n, F, squeeze = _pfb_args(x, P, M, window)
    buf, res = _pfb_out(out, squeeze, S, F, P if kind == COMPLEX else P // 2 + 1, torch.complex64, x.device)
    _check(lib().tina_pfb_batched(x.data_ptr(), S, n, P, M, window.data_ptr(), kind, prec,
                                  buf.data_ptr(), _stream_ptr(stream, x.device)))
    return res


def pfb_fft(x, P: int, M: int, window, out=None, stream=None):
    """tina_pfb_fft_batched: PFB with the factorised Fourier stage (complex P=1024 or real P=4096); same result as pfb()."""
    import torch
    kind, S, n, F, squeeze = _pfb_args(x, P, M, window)
    buf, res = _pfb_out(out, squeeze, S, F, P if kind == COMPLEX else P // 2 + 1, torch.complex64, x.device)
    _check(lib().tina_pfb_fft_batched(x.data_ptr(), S, n, P, M, window.data_ptr(), kind,
                                      buf.data_ptr(), _stream_ptr(stream, x.device)))
    return res


def pfb_fir(x, P: int, M: int, window, out=None, stream=None):
    """tina_pfb_fir_batched: subfilter stage only -> y [S, F, P] (dtype of x)."""
    kind, S, n, F, squeeze = _pfb_args(x, P, M, window)
    buf, res = _pfb_out(out, squeeze, S, F, P, x.dtype, x.device)
    _check(lib().tina_pfb_fir_batched(x.data_ptr(), S, n, P, M, window.data_ptr(), kind,
                                      buf.data_ptr(), _stream_ptr(stream, x.device)))
    return res


def pfb_host(x, P: int, M: int, window, prec: int = PREC_FP32, out=None, stream=None):
    """tina_pfb_batched_host: x, window, out are HOST tensors (pinned recommended); synchronous."""
    import torch
    if x.dim() == 1:
        x = x[None, :]
    if x.is_cuda or window.is_cuda or (out is not None and out.is_cuda):
        raise TypeError("pfb_host takes host tensors")
    kind = COMPLEX if x.dtype == torch.complex64 else REAL
    if kind == REAL and x.dtype != torch.float32:
        raise TypeError("x must be complex64 or float32")
    if x.dim() != 2 or not x.is_contiguous():
        raise ValueError("x must be a contiguous [S, n_samples] (or [n_samples]) tensor")
    if window.dtype != torch.float32 or not window.is_contiguous() or window.numel() != P * M:
        raise ValueError("window must be a contiguous float32 tensor with P*M entries")
    S, n = x.shape
    F = pfb_num_frames(n, P, M)
    NK = P if kind == COMPLEX else P // 2 + 1
    if out is None:
        out = torch.empty((S, max(F, 0), NK), dtype=torch.complex64, pin_memory=True)
    elif out.dtype != torch.complex64 or not out.is_contiguous() or tuple(out.shape) != (S, max(F, 0), NK):
        raise ValueError(f"out must be a contiguous complex64 host tensor of shape {(S, max(F, 0), NK)}")
    _check(lib().tina_pfb_batched_host(x.data_ptr(), S, n, P, M, window.data_ptr(), kind, prec,
                                       out.data_ptr(), _stream_ptr(stream)))
    return out
