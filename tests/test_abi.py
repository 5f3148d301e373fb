"""CPU-side checks of the C-ABI boundary (no GPU, no compute calls): the library builds, loads and exports every symbol
that include/tatrg.h declares; the entry points that validate arguments before touching the device return the
documented status codes; the product path never falls back to the CPU."""
import ctypes
import os
import re

import pytest

import paper_2507_21909_b200 as T

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2507_21909_b200 import build
    build.build()
    return T.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "tatrg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tatrg_[a-zA-Z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("tatrg_create", "tatrg_step", "tatrg_lnZ_per_site", "tatrg_singular_values", "tatrg_destroy"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib):
    raw = ctypes.CDLL(os.path.join(ROOT, "paper_2507_21909_b200", "libtatrg.so"))
    for name in declared_symbols():
        assert hasattr(raw, name), name
    # and the binding marshals exactly the declared set
    assert sorted(T.exported_symbols()) == declared_symbols()


def test_workspace_bytes_and_argument_validation(lib):
    assert lib.tatrg_workspace_bytes(1, 4) == 0          # D < 2
    assert lib.tatrg_workspace_bytes(4, -1) == 0
    assert lib.tatrg_workspace_bytes(64, 64) == 0        # D + p > 96
    w4, w32, w48 = (lib.tatrg_workspace_bytes(d, d) for d in (4, 32, 48))
    assert 0 < w4 < w32 < w48 < 170e9                    # config 5 fits one B200 (180 GB)
    assert w32 >= 8 * (32 ** 3 * 64 ** 2 + 6 * 32 ** 5)  # Xi (D^3 K^2) plus the 5-leg tensors
    h = ctypes.c_void_p()
    # every invalid argument is rejected before any CUDA call
    assert lib.tatrg_create(0.14, 0.0, 4, 4, 1, None, 0, ctypes.byref(h)) == T.EINVAL
    assert lib.tatrg_create(-1.0, 0.0, 4, 4, 1, ctypes.c_void_p(256), 1 << 40, ctypes.byref(h)) == T.EINVAL
    assert lib.tatrg_create(float("nan"), 0.0, 4, 4, 1, ctypes.c_void_p(256), 1 << 40, ctypes.byref(h)) == T.EINVAL
    assert lib.tatrg_create(0.14, 0.0, 1, 4, 1, ctypes.c_void_p(256), 1 << 40, ctypes.byref(h)) == T.EINVAL
    assert lib.tatrg_create(0.14, 0.0, 4, 4, 1, ctypes.c_void_p(257), 1 << 40, ctypes.byref(h)) == T.EINVAL   # alignment
    assert lib.tatrg_create(0.14, 0.0, 4, 4, 1, ctypes.c_void_p(256), 1024, ctypes.byref(h)) == T.ENOMEM
    assert lib.tatrg_create(0.14, 0.0, 4, 4, 1, ctypes.c_void_p(256), 1 << 40, None) == T.EINVAL
    assert lib.tatrg_step(None, None) == T.EINVAL
    assert lib.tatrg_set_option(None, 1, 1.0) == T.EINVAL
    v = lib.tatrg_lnZ_per_site(None)
    assert v != v                                        # NaN on error
    assert lib.tatrg_singular_values(None, 0, 4, None) == T.EINVAL
    assert lib.tatrg_eigh_work_bytes(0) == 0 and lib.tatrg_eigh_work_bytes(1024) >= 2 * 8 * 1024 * 1024
    assert lib.tatrg_svd_work_bytes(0, 3) == 0 and lib.tatrg_svd_work_bytes(8, 8) > 0
    assert lib.tatrg_dgemm(None, 0, 0, -1, 1, 1, 1.0, None, 1, None, 1, 0.0, None, 1, 1, 0, 0, 0) == T.EINVAL
    assert lib.tatrg_contract(None, b"ab,bc", None, None, None, None, None, None, 0) == T.EINVAL
    assert lib.tatrg_philox_raw(None, 0, 0, 0, 0, -1, None) == T.EINVAL


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(T.TatrgError):
        T.Tatrg(0.14, 0.0, 4, 4, 1)
    with pytest.raises(T.TatrgError):
        T.philox_raw(0, 0, 0, 0, 4)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2507_21909_b200")
    pat = re.compile(r"^\s*(import\s+oracle|from\s+oracle|from\s+\.+\s*oracle)|#include\s+[\"<].*oracle", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not pat.search(text), f
                assert "liborc_jacobi" not in text and "tatrg_oracle" not in text, f
