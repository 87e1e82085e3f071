"""CPU-only: the C-ABI library builds, loads, and exports every symbol include/bj.h declares;
without a GPU the compute entry points fail loudly (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "bj.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(bj_[a-zA-Z_0-9]+)\s*\(", txt)))


def test_header_declares_the_four_north_star_calls():
    syms = declared_symbols()
    for name in ("bj_setup", "bj_apply", "bj_op_apply", "bj_cond_estimate"):
        assert name in syms


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2410_02408_b200 import build as cuda_build
    from paper_2410_02408_b200 import binding
    lib = C.CDLL(cuda_build.build())
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/bj.h but not exported"
    assert sorted(binding.EXPORTS) == declared_symbols()
    L = binding.lib()
    for name in binding.EXPORTS:      # every entry point has its argument types declared (a bare int would pass as 32 bits)
        assert getattr(L, name).argtypes is not None, f"{name}: argtypes not set in binding.lib()"
    assert binding.lib().bj_strerror(0) == b"ok"
    assert binding.BJ_B_MAX == int(re.search(r"#define BJ_B_MAX (\d+)", open(os.path.join(ROOT, "include", "bj.h")).read()).group(1))


def test_no_cpu_fallback_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2410_02408_b200 import binding
    L = binding.lib()
    out = C.c_void_p()
    csr = binding.bj_csr_t(4, 4, 8, 8, 8)
    code = L.bj_setup(C.byref(csr), 2, C.byref(out))
    assert code == binding.BJ_ERR_CUDA and not out.value
    assert L.bj_setup(None, 2, C.byref(out)) == binding.BJ_ERR_INVALID_ARG
    assert L.bj_apply(None, None, None) == binding.BJ_ERR_INVALID_ARG


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2410_02408_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "bj_oracle" not in src, f
    orc = open(os.path.join(ROOT, "oracle", "bj_oracle.c")).read()
    assert "bj.h" not in orc and "cuda" not in orc.lower().replace("cuda library", "").replace("the cuda path", "")
