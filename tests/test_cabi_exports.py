"""CPU-side checks of the boundary: libsfft.so builds, loads and exports every symbol
include/sfft.h declares; without a CUDA device the product path fails loudly (no CPU fallback)."""
import ctypes
import re

import pytest
import torch

from conftest import ROOT


@pytest.fixture(scope="module")
def lib():
    from paper_2509_18544_b200 import build
    build.build()
    from paper_2509_18544_b200 import sfft
    return sfft.load_library()


def _declared():
    text = (ROOT / "include" / "sfft.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sfft_[a-z0-9_]+)\s*\(", text)))


def test_header_and_binding_agree(lib):
    from paper_2509_18544_b200 import sfft
    assert _declared() == sorted(sfft.SYMBOLS)


def test_every_declared_symbol_is_exported(lib):
    for name in _declared():
        assert hasattr(lib, name), name


def test_version_string(lib):
    from paper_2509_18544_b200 import sfft
    assert "sm_100a" in sfft.version()


def test_no_torch_types_in_header():
    text = (ROOT / "include" / "sfft.h").read_text()
    assert "torch" not in text.lower().replace("torch.cuda.current_stream", "")
    assert 'extern "C"' in text


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_fails_loudly_without_gpu(lib):
    from paper_2509_18544_b200 import SfftPlan
    with pytest.raises(RuntimeError):
        SfftPlan(64, 64, 3, 0, 0)
    h = ctypes.c_void_p()
    rc = lib.sfft_plan_create(ctypes.byref(h), 64, 64, 3, 0, 0)
    assert rc == -3 and not h.value  # SFFT_ERR_CUDA, never a CPU fallback


def test_product_never_imports_oracle():
    pkg = ROOT / "paper_2509_18544_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + list(pkg.rglob("*.h")):
        if "build/" in str(f):
            continue
        src = f.read_text()
        assert "import oracle" not in src and "from oracle" not in src and "sfft_oracle" not in src, f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c"):
            assert "paper_2509_18544_b200" not in f.read_text(), f
