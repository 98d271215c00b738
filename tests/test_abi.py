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


def declared_symbols(header="slidingattn.h"):
    text = (ROOT / "include" / header).read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ss_[a-z_]+)\s*\(", text)))


# the product boundary is exactly this list (plus lifetime / status helpers)
SECTION_8B = {"ss_create", "ss_destroy", "ss_workspace_bytes", "ss_kv_append", "ss_mixed_attention",
              "ss_poll_device_error", "ss_status_string"}


def test_header_declares_the_two_path_calls():
    syms = declared_symbols()
    assert SECTION_8B <= set(syms)
    assert not any(s.startswith("ss_debug") or "timing" in s or "worklist" in s for s in syms), \
        "measurement / debug aids belong in slidingattn_debug.h"


def test_library_exports_every_declared_symbol(lib):
    from paper_2606_05933_b200 import binding
    for header in ("slidingattn.h", "slidingattn_debug.h"):
        for name in declared_symbols(header):
            assert hasattr(lib, name), f"{name} declared in {header} but not exported"
    assert sorted(binding.EXPORTS) == declared_symbols()
    assert sorted(binding.DEBUG_EXPORTS) == declared_symbols("slidingattn_debug.h")


def test_version_and_status_strings(lib):
    assert lib.ss_version() == 200
    assert lib.ss_status_string(0) == b"SS_OK"
    assert lib.ss_status_string(-1) == b"SS_ERR_INVALID_ARG"
    assert lib.ss_status_string(-2) == b"SS_ERR_WORKSPACE_TOO_SMALL"
    assert lib.ss_status_string(-3) == b"SS_ERR_UNSUPPORTED_DEVICE"
    assert lib.ss_status_string(-6) == b"SS_ERR_DEVICE_CHECK"


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
    assert lib.ss_poll_device_error(None, None) == -1 and lib.ss_reset(None, None) == -1
    assert lib.ss_set_kv_scales(None, None, None) == -1
    bad = ss_config(32, 8, 128, 16, 64, 4, 64, 8, 4)         # unknown flag bit
    assert lib.ss_create(ctypes.byref(h), ctypes.byref(bad), 256, 512) == -1
    bad = ss_config(8, 8, 64, 16, 64, 4, 64, 8, 2)           # SS_FLAG_KV_FP8 needs head_dim 128
    assert lib.ss_create(ctypes.byref(h), ctypes.byref(bad), 256, 512) == -1
    bad = ss_config(64, 8, 128, 16, 64, 2048, 2 ** 31 - 1, 2 ** 26)   # worst-case item count overflows int32
    assert lib.ss_create(ctypes.byref(h), ctypes.byref(bad), 256, 512) == -1


def test_binding_refuses_wrong_dtypes_and_shapes():
    """torch's default int64 index tensors must not reach the raw-pointer ABI."""
    import torch
    from paper_2606_05933_b200 import binding
    with pytest.raises(binding.SlidingAttnError, match="int32"):
        binding._want(torch.zeros(4, dtype=torch.int64), "ctx_lens", torch.int32, cuda=False)
    with pytest.raises(binding.SlidingAttnError, match="contiguous"):
        binding._want(torch.zeros(4, 4, dtype=torch.int32)[:, ::2], "block_table", torch.int32, cuda=False)
    with pytest.raises(binding.SlidingAttnError, match="shape"):
        binding._want(torch.zeros(5, dtype=torch.int32), "query_start_loc", torch.int32, cuda=False, shape=(4,))
    with pytest.raises(binding.SlidingAttnError, match="CUDA"):
        binding._want(torch.zeros(4, dtype=torch.int32), "ctx_lens", torch.int32, cuda=True)


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
