"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every entry
point include/slidingattn.h declares; the binding marshals the same names; no compute calls here."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2606_05933_b200 import build, binding
    build.build()
    return binding.load()


def declared_symbols():
    text = (ROOT / "include" / "slidingattn.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ss_[a-z_]+)\s*\(", text)))


def test_header_declares_the_two_path_calls():
    syms = declared_symbols()
    assert "ss_kv_append" in syms and "ss_mixed_attention" in syms and len(syms) >= 8


def test_library_exports_every_declared_symbol(lib):
    from paper_2606_05933_b200 import binding
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in slidingattn.h but not exported"
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_version_and_status_strings(lib):
    assert lib.ss_version() == 100
    assert lib.ss_status_string(0) == b"SS_OK"
    assert lib.ss_status_string(-1) == b"SS_ERR_INVALID_ARG"
    assert lib.ss_status_string(-2) == b"SS_ERR_WORKSPACE_TOO_SMALL"
    assert lib.ss_status_string(-3) == b"SS_ERR_UNSUPPORTED_DEVICE"


def test_null_arguments_are_rejected_without_a_device(lib):
    from paper_2606_05933_b200.binding import ss_config
    h = ctypes.c_void_p()
    assert lib.ss_create(None, None, None, None) == -1
    cfg = ss_config(32, 8, 128, 16, 64, 4, 64, 8)
    assert lib.ss_create(ctypes.byref(h), ctypes.byref(cfg), None, None) == -1
    bad = ss_config(32, 8, 96, 16, 64, 4, 64, 8)            # head_dim not in {64,128}
    assert lib.ss_create(ctypes.byref(h), ctypes.byref(bad), 256, 512) == -1
    bad = ss_config(32, 5, 128, 16, 64, 4, 64, 8)            # Hq % Hkv != 0
    assert lib.ss_create(ctypes.byref(h), ctypes.byref(bad), 256, 512) == -1
    bad = ss_config(32, 8, 128, 32, 64, 4, 64, 8)            # page size != 16
    assert lib.ss_create(ctypes.byref(h), ctypes.byref(bad), 256, 512) == -1
    assert lib.ss_kv_append(None, None, None, None, None, None, 1, 1, None) == -1
    assert lib.ss_workspace_bytes(None) == 0


def test_binding_refuses_cpu_tensors(lib):
    import torch
    from paper_2606_05933_b200 import binding
    k = torch.zeros(4, 2, 16, 64, dtype=torch.bfloat16)
    with pytest.raises(binding.SlidingAttnError):
        binding.SlidingAttn(4, 2, 64, k, k.clone(), 4, 64, 4)


def test_product_does_not_import_oracle():
    """The product path may not import, include or execute anything under oracle/."""
    pat = re.compile(r"^\s*(import\s+oracle|from\s+oracle)|#include\s*[<\"].*oracle|liboracle", re.M)
    for p in (ROOT / "paper_2606_05933_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            assert not pat.search(p.read_text()), p
