"""CPU-side checks of the boundary: libqk.so builds (nvcc cross-compiles for sm_100a without a
GPU), loads, and exports every symbol include/qk.h declares; argument validation that needs no
device; the Python binding refuses to run without CUDA (there is no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

from paper_2110_01792_b200 import binding as B
from paper_2110_01792_b200 import build as qkbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    qkbuild.build()
    return B.lib()


def _declared():
    text = open(os.path.join(ROOT, "include", "qk.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qk_[A-Za-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 25
    raw = C.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), "include/qk.h declares %s but libqk.so does not export it" % n
    assert sorted(B.EXPORTS) == names, "binding.EXPORTS and include/qk.h disagree"


def test_binding_has_every_entry_point():
    for n in _declared():
        assert n in B.EXPORTS
        if n not in ("qk_init", "qk_free", "qk_state_bytes", "qk_bind_storage", "qk_version",
                     "qk_kernel_class_count", "qk_kernel_class_name", "qk_fp64_probe", "qk_selftest_divsqrt",
                     "qk_noalloc_setup", "qk_noalloc_max_cells", "qk_cfl_dt_noalloc"):
            assert hasattr(B.Context, n), n


def test_state_bytes(lib):
    n = 32
    cells = (n + 8) ** 3
    b = lib.qk_state_bytes(n, n, n)
    assert b >= 17 * cells * 8          # 11 state + 5 stage + chi
    assert lib.qk_state_bytes(0, 4, 4) == 0
    # 512^3 (BASELINE.json configs[4]) fits one B200's 180 GB with room to spare
    assert lib.qk_state_bytes(512, 512, 512) < 60e9


def test_version_and_class_names(lib):
    assert b"sm_100a" in lib.qk_version()
    n = lib.qk_kernel_class_count()
    names = [lib.qk_kernel_class_name(k).decode() for k in range(n)]
    assert "exchange" in names and "fill_boundary" in names and len(set(names)) == n


def test_null_and_invalid_arguments(lib):
    h = C.c_void_p()
    assert lib.qk_init(0, 4, 4, 0.1, 1.4, 0.0, 0.0, 0, C.byref(h)) == B.QK_EINVAL
    assert lib.qk_init(4, 4, 4, -1.0, 1.4, 0.0, 0.0, 0, C.byref(h)) == B.QK_EINVAL
    assert lib.qk_init(4, 4, 4, 0.1, 1.0, 0.0, 0.0, 0, C.byref(h)) == B.QK_EINVAL
    assert lib.qk_init(4, 4, 4, 0.1, 1.4, 0.0, 0.0, 7, C.byref(h)) == B.QK_EINVAL
    assert lib.qk_free(None) == B.QK_EINVAL
    assert lib.qk_hydro_step(None, 0.1) == B.QK_EINVAL
    assert lib.qk_launch_count(None) == -1


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(B.QkError):
        B.Context(8, 8, 8, 0.1, 1.4)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2110_01792_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "qk_oracle.h" not in text and "from oracle" not in text, f
