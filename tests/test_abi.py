"""CPU-side checks of the C-ABI boundary: liblloid.so builds, loads and exports every symbol that
include/lloid.h declares; argument validation that needs no GPU.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2410_16416_b200 import build, binding
    build.build()
    return binding.lib()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "lloid.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lloid_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    names = declared_functions()
    for must in ("lloid_bank_create", "lloid_bank_upload_slice", "lloid_bank_finalize", "lloid_filter",
                 "lloid_filter_host", "lloid_reset", "lloid_destroy", "lloid_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    from paper_2410_16416_b200 import binding
    raw = C.CDLL(binding.LIB_PATH)
    for name in declared_functions():
        assert hasattr(raw, name), f"{name} declared in include/lloid.h but not exported"
        assert name in binding.EXPORTS, f"{name} has no Python binding"
    assert sorted(binding.EXPORTS) == declared_functions()


def test_struct_layouts_match_header():
    from paper_2410_16416_b200 import binding as lb
    assert C.sizeof(lb.lloid_trigger_t) == 32
    assert C.sizeof(lb.lloid_bank_config_t) == 40
    assert C.sizeof(lb.lloid_bin_desc_t) == 16
    assert C.sizeof(lb.lloid_slice_desc_t) == 24
    assert lb.lloid_trigger_t.sample.offset == 16 and lb.lloid_trigger_t.snr_re.offset == 24


def test_check_count_and_version(lib):
    from paper_2410_16416_b200 import binding as lb
    assert lb.lloid_check_count(3, 3) == lb.LLOID_OK
    assert lb.lloid_check_count(4, 3) == lb.LLOID_EOVERFLOW
    assert "overflow" in lb.lloid_last_error()
    assert "sm_100a" in lb.lloid_version()


def test_create_rejects_bad_arguments_without_touching_the_gpu(lib):
    from paper_2410_16416_b200 import binding as lb
    out = C.c_void_p()
    assert lib.lloid_bank_create(C.byref(out), None, None, None) == lb.LLOID_EINVAL
    cfg = lb.lloid_bank_config_t(1, 1, 2048, 2048, 4.0, 16, 8, lb.LLOID_F32, 0, 0)
    bins = (lb.lloid_bin_desc_t * 1)(lb.lloid_bin_desc_t(4, 1, 128))
    sl = (lb.lloid_slice_desc_t * 1)(lb.lloid_slice_desc_t(2048, 128, 8, 0, 0))
    ptrs = (C.POINTER(lb.lloid_slice_desc_t) * 1)(C.cast(sl, C.POINTER(lb.lloid_slice_desc_t)))
    for field, bad in (("n_bins", 0), ("peak_window", 100), ("k_up", 4), ("precision", 7), ("max_chunk", 100)):
        c2 = lb.lloid_bank_config_t.from_buffer_copy(cfg)
        setattr(c2, field, bad)
        assert lib.lloid_bank_create(C.byref(out), C.byref(c2), bins, ptrs) == lb.LLOID_EINVAL, field
        assert lb.lloid_last_error()


def test_no_cpu_fallback_without_a_gpu(lib):
    """On a box without a CUDA device bank creation must fail with LLOID_ECUDA (never fall back)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2410_16416_b200 import binding as lb, workloads as wl
    w = wl.toy()
    with pytest.raises(lb.LloidError) as e:
        lb.Bank(w, lb.LLOID_F32)
    assert e.value.code == lb.LLOID_ECUDA


def test_product_code_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2410_16416_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f), errors="ignore").read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
    src = open(os.path.join(ROOT, "oracle", "lloid_oracle.py")).read()
    assert "paper_2410_16416_b200" not in re.sub(r'""".*?"""', "", src, flags=re.S)
