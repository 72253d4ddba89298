"""CPU-only checks of the boundary: the C-ABI library builds/loads and exports every symbol include/fdtd.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared(headers=("fdtd.h", "fdtd_bench.h")):
    names = set()
    for h in headers:
        txt = open(os.path.join(ROOT, "include", h)).read()
        txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
        names |= set(re.findall(r"\b(fdtd_[a-z_0-9]+)\s*\(", txt))
    return sorted(names)


def test_bench_instrumentation_is_not_in_the_product_header():
    product = _declared(("fdtd.h",))
    assert "fdtd_profile_kernel" not in product and "fdtd_launch_count" not in product
    assert set(_declared(("fdtd_bench.h",))) == {"fdtd_profile_kernel", "fdtd_launch_count", "fdtd_debug_guard_check"}


def test_header_declares_the_four_north_star_calls():
    d = _declared()
    for name in ("fdtd_create", "fdtd_forward", "fdtd_reverse", "fdtd_store_bytes"):
        assert name in d


def test_library_exports_every_declared_symbol():
    from paper_2603_24027_b200 import build, fdtd
    path = build.build()
    L = ctypes.CDLL(path)
    decl = _declared()
    assert len(decl) >= 25
    for name in decl:
        assert hasattr(L, name), f"{name} declared in include/fdtd.h but not exported"
    assert sorted(fdtd.EXPORTED) == decl


def test_no_cpu_fallback_without_cuda():
    import torch
    from paper_2603_24027_b200 import fdtd
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(fdtd.FdtdError):
        fdtd.Sim(torch.ones(8, 8, 8), 20e-9, 3.8e-17, 2)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2603_24027_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "fdtd_oracle" not in src, f
    for f in ("fdtd_oracle.cpp", "fdtd_oracle.py"):
        src = open(os.path.join(ROOT, "oracle", f)).read()
        assert "import paper_2603_24027_b200" not in src and "from paper_2603_24027_b200" not in src and "libfdtd_b200" not in src
