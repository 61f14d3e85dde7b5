"""The boundary: libwhiflash.so builds without a GPU (nvcc cross-compiles sm_100a), loads, and exports every function
include/whiflash.h declares; the Python binding lists the same names; without a CUDA device the product path fails
loudly (no CPU fallback).  No compute call is made here."""

import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "whiflash.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)                       # drop comments
    names = re.findall(r"^\s*(?:const\s+)?(?:int|size_t|char\s*\*|int32_t\s*\*|int64_t)\s*\*?\s*(wf_[a-z0-9_]+)\s*\(", src, flags=re.M)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2606_07710_b200 import build
    return build.build()


def test_header_declares_the_hot_path_calls():
    names = _declared()
    for must in ("wf_verify_attn", "wf_accept_entropy_route", "wf_kv_only_prefill", "wf_lazy_catchup_enqueue",
                 "wf_lazy_catchup_flush", "wf_lazy_catchup_round", "wf_kv_create", "wf_kv_reserve", "wf_kv_release_seq",
                 "wf_neural_route", "wf_ctx_create", "wf_poll_status", "wf_last_error"):
        assert must in names, must


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    missing = [n for n in _declared() if not hasattr(lib, n)]
    assert not missing, missing


def test_binding_lists_exactly_the_declared_symbols(lib_path):
    from paper_2606_07710_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()
    assert all(hasattr(binding.lib, n) for n in binding.EXPORTS)


def test_no_cpu_fallback_without_a_device(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2606_07710_b200 import binding
    with pytest.raises(binding.WhiFlashError):
        binding.Ctx(0)
