"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/hft.h declares, and its
argument validation / host-only entry points behave (no compute calls without a GPU)."""
import ctypes as C
import os
import re

import pytest

from helpers import ROOT


@pytest.fixture(scope="module")
def lib():
    from paper_2501_06377_b200 import build
    path = build.build()
    return C.CDLL(path)


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "hft.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hft_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    syms = declared_symbols()
    assert len(syms) >= 18
    for s in syms:
        assert hasattr(lib, s), s
    from paper_2501_06377_b200 import hft
    assert sorted(hft.EXPORTS) == syms


def test_workspace_bytes_and_argument_errors(lib):
    from paper_2501_06377_b200 import hft
    n = hft.workspace_bytes(1024, 2048, 64, "f64")
    assert n == 6 * 64 * 1026 * 2048 * 8
    assert hft.workspace_bytes(1024, 2048, 64, "f32") == n // 2
    # pitch padding: 1023 fp64 columns -> 1024
    assert hft.workspace_bytes(510, 1023, 1, "f64") == 6 * 512 * 1024 * 8
    g = hft.hft_grid(4, 2048, 1, 0, 1.0)
    out = C.c_size_t()
    assert lib.hft_workspace_bytes(C.byref(g), 1, None, C.byref(out)) == -1
    assert lib.hft_workspace_bytes(None, 1, None, C.byref(out)) == -1
    h = C.c_void_p()
    lib.hft_create.argtypes = hft._lib.hft_create.argtypes
    assert lib.hft_create(None, 1, None, None, None, 0, None, C.byref(h)) == -1
    assert lib.hft_step(None, 1, C.c_double(1.0)) == -1
    lib.hft_error_string.restype = C.c_char_p
    assert lib.hft_error_string(0) == b"ok" and b"workspace" in lib.hft_error_string(-2)


def test_create_fails_loudly_without_a_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2501_06377_b200 import hft
    with pytest.raises(hft.HftError):
        hft.Context(64, 128, [[500.0, 0, 0, 0, 0, 0, 0]])
    g = hft.hft_grid(64, 128, 1, 0, 1.0)
    p = (hft.hft_params * 1)(hft.hft_params(500.0, 0, 0, 0, 0, 0, 0))
    h = C.c_void_p()
    rc = hft._lib.hft_create(C.byref(g), 1, p, None, C.c_void_p(256), hft.workspace_bytes(64, 128, 1), None, C.byref(h))
    assert rc == -6 and not h.value


def test_product_never_imports_the_oracle():
    """The product path must not route through oracle/ (and the oracle must not import the CUDA package)."""
    pkg = os.path.join(ROOT, "paper_2501_06377_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                for needle in ("import oracle", "from oracle", "sft_oracle", "oracle/", "oracle."):
                    assert needle not in src, (dirpath, f, needle)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2501_06377_b200" not in src and "from paper_2501_06377_b200" not in src
            assert "hft.h" not in src and "csrc" not in src.replace("paper_2501_06377_b200/csrc/", "")


def test_workspace_grows_with_the_optional_rows(lib):
    """hft_options.flow_attenuation reserves 6 more field arrays, hft_options.rfe 2 more; invalid options are refused."""
    from paper_2501_06377_b200 import hft
    one = 4 * 66 * 128 * 8          # n_real x (n_theta + 2) x pitch x sizeof(double)
    base = hft.workspace_bytes(64, 128, 4, "f64")
    assert base == 6 * one
    opt = hft.hft_options(2, 4, 3, 0, 0, 0, 0, 1)
    assert hft.workspace_bytes(64, 128, 4, "f64", opt) == 12 * one
    opt = hft.hft_options(2, 4, 3, 0, 0, 1, 1, 1)
    assert hft.workspace_bytes(64, 128, 4, "f64", opt) == 14 * one
    opt = hft.hft_options(2, 4, 3, 0, 0, 1, 1, 1, 1)
    assert hft.workspace_bytes(64, 128, 4, "f64", opt) == 15 * one
    for bad in (hft.hft_options(5, 4, 3, 0, 0, 0, 0, 0), hft.hft_options(2, 2, 3, 0, 0, 0, 0, 0), hft.hft_options(2, 4, 3, 1, 0, 0, 0, 0),
                hft.hft_options(2, 4, 3, 0, 3, 0, 0, 0), hft.hft_options(2, 4, 3, 0, 0, 2, 0, 0), hft.hft_options(2, 4, 3, 0, 0, 0, 0, 7),
                hft.hft_options(2, 4, 3, 0, 0, 0, 0, 0, 2)):
        with pytest.raises(hft.HftError):
            hft.workspace_bytes(64, 128, 4, "f64", bad)
