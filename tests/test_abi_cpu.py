"""CPU-only checks of the boundary: libtina.so builds, loads and exports every symbol that
include/tina.h declares; host-side argument validation (no compute calls without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2408_16551_b200 import build, binding
    build.build()
    return binding.lib()


def test_exports_match_header(L):
    hdr = open(os.path.join(ROOT, "include", "tina.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(tina_[a-z0-9_]+)\s*\(", hdr))
    assert {"tina_fir", "tina_dft", "tina_pfb"} <= declared
    from paper_2408_16551_b200 import binding
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name


def test_num_frames_and_strings(L):
    assert L.tina_pfb_num_frames(65584, 16, 4) == 4096
    assert L.tina_pfb_num_frames((8192 + 15) * 1024, 1024, 16) == 8192
    assert L.tina_pfb_num_frames(1 << 27, 4096, 8) == 32761
    assert L.tina_pfb_num_frames(48, 16, 4) == 0
    assert L.tina_status_string(0) == b"TINA_OK"
    assert L.tina_status_string(4) == b"TINA_ERR_ALIGNMENT"
    assert L.tina_version() >= 100
    assert L.tina_launch_count() == 0 or L.tina_launch_count() > 0


def test_validation_without_gpu(L):
    buf = (ctypes.c_char * 4096)()
    a = ctypes.addressof(buf)
    a16 = (a + 15) & ~15
    assert L.tina_fir(None, a16, a16 + 64, 1, 10, 2, None) == 1            # NULL_POINTER
    assert L.tina_fir(a16, a16, a16 + 64, 1, 3, 5, None) == 2              # L < M
    assert L.tina_fir(a16, a16, a16 + 64, 0, 10, 2, None) == 2
    assert L.tina_fir(a16 + 4, a16, a16 + 64, 1, 10, 2, None) == 4         # ALIGNMENT
    assert L.tina_fir(a16, a16, a16 + 64, 1, 10000, 5000, None) == 3       # UNSUPPORTED M
    assert L.tina_dft(a16, a16, 1, 8, 0, 0, None) == 2                     # in-place
    assert L.tina_dft(a16, a16 + 64, 1, 1, 0, 0, None) == 2                # N < 2
    assert L.tina_dft(a16, a16 + 64, 1, 16384, 0, 0, None) == 3
    assert L.tina_pfb(a16, 48, 16, 4, a16 + 512, 0, 0, a16 + 1024, None) == 2   # F = 0
    assert L.tina_pfb(a16, 100, 5, 1, a16 + 512, 1, 0, a16 + 1024, None) == 2   # odd P real
    assert L.tina_pfb(a16, 1000, 16, 100, a16 + 512, 0, 0, a16 + 1024, None) == 3  # M > 64
    assert L.tina_pfb(a16, 64, 16, 4, None, 0, 0, a16 + 1024, None) == 1
    assert L.tina_pfb_batched(a16, 2, 65, 16, 4, a16 + 512, 0, 0, a16 + 1024, None) == 4  # odd stride
    assert b"n_samples" in L.tina_last_error()
