"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/leb.h
declares, and the Python binding names the same calls.  No compute call is made (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "leb.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2607_01203_b200 import build, leb
    build.build()
    return leb.load_library()


def _declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(leb_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for must in ("leb_analytic_fwd", "leb_nn_fwd", "leb_vjp", "leb_zonotope_inflate"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in _declared_symbols():
        assert hasattr(lib, name), name


def test_binding_lists_the_same_symbols(lib):
    from paper_2607_01203_b200 import leb
    assert sorted(leb.EXPORTS) == _declared_symbols()
    for name in ("leb_analytic_fwd", "leb_nn_fwd", "leb_vjp", "leb_zonotope_inflate", "leb_set_mlp", "leb_set_analytic"):
        assert hasattr(leb.Context, name)


def test_status_strings(lib):
    lib.leb_status_str.restype = ctypes.c_char_p
    assert lib.leb_status_str(0) == b"ok"
    assert b"unsupported" in lib.leb_status_str(5)


def test_null_arguments_are_rejected_without_a_device(lib):
    # argument errors are synchronous and need no GPU
    assert lib.leb_create(None, 0) == 1                      # LEB_ERR_ARG
    assert lib.leb_set_analytic(None, None) == 1
    assert lib.leb_launch_count(None) == 0


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_01203_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "from oracle" not in text and "import oracle" not in text, f
                assert "pbh_oracle" not in text and "nn_oracle" not in text, f


def test_no_cpu_fallback_without_cuda():
    import torch
    from paper_2607_01203_b200 import leb
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError):
        leb.Context(0)
