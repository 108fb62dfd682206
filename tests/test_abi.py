"""CPU-only checks of the boundary: libbang.so builds for sm_100a, loads, and exports every symbol that
include/bang.h declares; argument validation that needs no device.  No compute calls are made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libbang():
    from paper_2205_06819_b200 import build, bang
    build.build()
    return bang.lib()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "bang.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bang_[a-z_]+)\s*\(", src)))


def test_header_declares_the_two_calls_of_the_problem_statement():
    syms = _declared_symbols()
    for name in ("bang_create", "bang_set_data", "bang_model_maps", "bang_loglike", "bang_destroy",
                 "bang_strerror", "bang_last_error"):
        assert name in syms


def test_library_exports_every_declared_symbol(libbang):
    from paper_2205_06819_b200 import bang
    syms = _declared_symbols()
    assert len(syms) >= 10
    for name in syms:
        assert hasattr(libbang, name), name
    assert sorted(bang.EXPORTS) == syms          # the Python binding mirrors the ABI one to one


def test_strerror_is_static_text(libbang):
    from paper_2205_06819_b200 import bang
    assert libbang.bang_strerror(0) == b"success"
    for code in (bang.EINVAL, bang.ENOMEM, bang.ECUDA, bang.ENODATA):
        assert len(libbang.bang_strerror(code)) > 0
    assert libbang.bang_last_error(None) == b""
    assert libbang.bang_launch_count(None) == 0
    libbang.bang_destroy(None)                   # NULL is allowed


def test_create_rejects_bad_configurations_before_touching_a_device(libbang):
    from paper_2205_06819_b200 import bang
    h = C.c_void_p(123)
    good_g = bang.Grid(16, 16, 1.0, 2, 50.0)
    good_p = bang.Psf(1.0, 3.0)
    good_m = bang.Model(bang.BULGE | bang.DISC1, 0, 0, 32, bang.FP64)

    def create(g, p, m):
        rc = libbang.bang_create(C.byref(h), C.byref(g), C.byref(p), C.byref(m), 0, None)
        assert h.value is None                    # *out is NULL on failure
        return rc

    assert create(bang.Grid(0, 16, 1.0, 2, 50.0), good_p, good_m) == bang.EINVAL
    assert create(bang.Grid(16, 16, 1.0, 5, 50.0), good_p, good_m) == bang.EINVAL      # s > 4
    assert create(bang.Grid(16, 16, -1.0, 2, 50.0), good_p, good_m) == bang.EINVAL
    assert create(good_g, bang.Psf(-1.0, 3.0), good_m) == bang.EINVAL
    assert create(good_g, bang.Psf(5.0, 3.0), good_m) == bang.EINVAL                   # footprint > 13 pixels
    assert create(good_g, good_p, bang.Model(bang.HALO, 0, 0, 32, bang.FP64)) == bang.EINVAL   # nothing luminous
    assert create(good_g, good_p, bang.Model(3, 0, 7, 32, bang.FP64)) == bang.EINVAL
    assert create(good_g, good_p, bang.Model(3, 0, 0, 0, bang.FP64)) == bang.EINVAL
    assert create(good_g, good_p, bang.Model(3, 0, 0, 32, 9)) == bang.EINVAL
    assert libbang.bang_create(None, C.byref(good_g), C.byref(good_p), C.byref(good_m), 0, None) == bang.EINVAL


def test_product_path_fails_loudly_without_cuda():
    import torch
    from paper_2205_06819_b200 import bang, workloads as W
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError):
        bang.Context(W.config(1))
    # and straight through the ABI: no device -> BANG_ECUDA, never a CPU result
    h = C.c_void_p()
    g, p, m = bang.Grid(16, 16, 1.0, 2, 50.0), bang.Psf(1.0, 3.0), bang.Model(3, 0, 0, 32, bang.FP64)
    assert bang.lib().bang_create(C.byref(h), C.byref(g), C.byref(p), C.byref(m), 0, None) == bang.ECUDA


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2205_06819_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "bang_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f
    for f in ("bang_oracle.cpp", "bang_oracle.py"):
        txt = open(os.path.join(ROOT, "oracle", f)).read()
        assert "libbang.so" not in txt and "csrc" not in txt and "bang.h" not in txt
