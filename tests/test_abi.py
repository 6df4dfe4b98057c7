"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/mhd.h declares; argument errors are reported without touching a device."""
import ctypes
import os
import re
import shutil

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mhd.h")


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mhd_[a-z_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2402_05240_b200 import build
    if not os.path.exists(build.LIB):
        if shutil.which("nvcc") is None and not os.path.exists("/usr/local/cuda/bin/nvcc"):
            pytest.skip("nvcc not available and libmhd.so not built")
    return build.build()


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("mhd_init", "mhd_set_state", "mhd_compute_dt", "mhd_step", "mhd_get_state"):
        assert name in syms


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for name in declared_symbols():
        assert hasattr(L, name), name


def test_argument_errors_without_a_device(libpath):
    L = ctypes.CDLL(libpath)
    L.mhd_workspace_bytes.restype = ctypes.c_size_t
    L.mhd_last_error.restype = ctypes.c_char_p
    assert L.mhd_workspace_bytes(0, 4, 4, 1) == 0
    assert L.mhd_workspace_bytes(4, 4, 4, 5) == 0
    # 40 arrays of pitch 40 (4 + 32 + 4) * 40 * 40 doubles, PLMC ng = 4
    nbytes = L.mhd_workspace_bytes(32, 32, 32, 1)
    assert nbytes >= 40 * 40 * 40 * 40 * 8
    assert L.mhd_step(ctypes.c_double(0.1)) == -2        # not initialised
    assert L.mhd_set_boundary(0, 1) == -2
    assert L.mhd_init(0, 1, 1, ctypes.c_double(1.4), 1) == -1
    assert b"bad argument" in L.mhd_last_error()
    assert L.mhd_finalize() == 0


def test_binding_has_no_cpu_fallback():
    """The product path must fail loudly without CUDA, never route through the oracle."""
    src = open(os.path.join(ROOT, "paper_2402_05240_b200", "mhd.py")).read()
    assert "oracle" not in src.replace("no CPU fallback", "")
    import torch
    if not torch.cuda.is_available():
        from paper_2402_05240_b200 import mhd
        with pytest.raises(mhd.MhdError):
            mhd.Mhd(8, 8, 8, 5.0 / 3.0)
