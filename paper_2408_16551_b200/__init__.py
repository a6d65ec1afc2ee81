"""paper_2408_16551_b200 -- B200-native FIR / DFT / polyphase-filter-bank library (TINA hot path).

Thin Python binding over the C ABI in ``include/tina.h`` (``libtina.so``, hand-written CUDA
for sm_100a).  PyTorch is used only for device memory and streams.
"""
from .binding import (TinaError, fir, fir_multi, unfold, mul, add, summation, summation_static, matmul, dft, pfb, pfb_fft, pfb_fir, pfb_host, pfb_num_frames, launch_count,
                      last_path, last_kernel, last_issued_ratio, clear_plan_cache, reload_options, build_is_dev, probe_peak, version, lib, COMPLEX, REAL, PREC_FP32, PREC_BF16, PREC_FP16)

__all__ = ["TinaError", "fir", "fir_multi", "unfold", "mul", "add", "summation", "summation_static", "matmul", "dft", "pfb", "pfb_fft", "pfb_fir", "pfb_host", "pfb_num_frames", "launch_count",
           "last_path", "last_kernel", "last_issued_ratio", "clear_plan_cache", "reload_options", "build_is_dev", "probe_peak", "version", "lib", "COMPLEX", "REAL", "PREC_FP32", "PREC_BF16", "PREC_FP16"]
