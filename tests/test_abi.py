"""CPU-side checks of the boundary: libqw.so builds for sm_100a without a GPU, loads, exports every
symbol include/qw.h declares, and — with no device — fails loudly instead of falling back."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    text = open(os.path.join(ROOT, "include", "qw.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qw_[a-z_]+)\s*\(", text)))


def test_header_and_binding_agree(qw):
    assert header_symbols() == sorted(qw.SYMBOLS)


def test_library_exports_every_declared_symbol(qw):
    lib = qw.load()
    for name in header_symbols():
        assert hasattr(lib, name), name


def test_header_is_plain_c(tmp_path):
    """include/qw.h compiles as C (no torch / C++ types in the boundary)."""
    src = tmp_path / "t.c"
    src.write_text('#include "qw.h"\nint main(void){ qw_sim *s = 0; (void)s; return QW_OK; }\n')
    import subprocess
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                           "-c", str(src), "-o", str(tmp_path / "t.o")])


def test_argument_errors_do_not_need_a_device(qw):
    lib = qw.load()
    h = ctypes.c_void_p()
    ext = (ctypes.c_int64 * 2)(8, 8)
    assert lib.qw_create(3, ext, 6, qw.QW_C128, qw.QW_OPEN, ctypes.byref(h)) == qw.QW_EINVAL
    assert b"dim" in lib.qw_last_error()
    assert lib.qw_create(1, ext, 4, qw.QW_C128, qw.QW_OPEN, ctypes.byref(h)) == qw.QW_EINVAL   # coin_dim != 2*dim
    assert lib.qw_create(2, ext, 4, 7, qw.QW_OPEN, ctypes.byref(h)) == qw.QW_EINVAL
    assert lib.qw_create(2, ext, 4, qw.QW_C64, 5, ctypes.byref(h)) == qw.QW_EINVAL
    bad = (ctypes.c_int64 * 2)(8, 0)
    assert lib.qw_create(2, bad, 4, qw.QW_C64, qw.QW_OPEN, ctypes.byref(h)) == qw.QW_EINVAL
    assert lib.qw_create_batch(0, 1, ext, 2, qw.QW_C64, qw.QW_OPEN, ctypes.byref(h)) == qw.QW_EINVAL
    assert lib.qw_step(None, 1) == qw.QW_EINVAL
    assert lib.qw_destroy(None) == qw.QW_OK


def test_no_cpu_fallback_without_a_device(qw):
    """On a box without a GPU creating a handle must fail with QW_ECUDA — never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(qw.QwError) as ei:
        qw.qw_create(1, [16], 2, qw.QW_C128, qw.QW_PERIODIC)
    assert ei.value.code == qw.QW_ECUDA


def test_product_does_not_import_the_oracle():
    """The package and its sources never reference oracle/ (parity would be void otherwise)."""
    pkg = os.path.join(ROOT, "paper_1003_3779_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in dirpath.split(os.sep)[-1:]:
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "qw_oracle" not in text and "qwo_" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libqw.so" not in text and "csrc" not in text.replace("paper_1003_3779_b200/csrc", ""), f
            assert "import paper_1003_3779_b200" not in text and "from paper_1003_3779_b200" not in text, f


def test_workload_builders_shapes():
    from paper_1003_3779_b200 import inputs as qi
    w = qi.k0()
    assert w.extents == (201,) and w.steps == 100 and w.boundary == qi.OPEN
    w = qi.k1(log2_sites=10, steps=5)
    assert w.state.shape == (1, 1024, 2) and abs(np.sum(np.abs(w.state) ** 2) - 1) < 1e-14
    w = qi.k1(log2_sites=10, steps=5, dtype=np.complex64)
    assert w.state.dtype == np.complex64 and w.coin.dtype == np.complex64
    w = qi.k2(half=8)
    assert w.extents == (17, 17) and w.steps == 8
    w = qi.k3(extent=16, steps=3, coin="dft")
    assert w.state.shape == (1, 256, 4) and w.dtype == np.complex64
    w = qi.k4(batch=3, half=4)
    assert w.coin.shape == (3, 2, 2) and w.phases.shape == (3, 9)
    mode, coin = w.general_coin_f64()
    assert mode == qi.COIN_PER_SITE and coin.shape == (3, 9, 2, 2)
