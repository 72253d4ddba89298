"""The boundary as a C ABI: a plain C99 translation unit (tests/abi_c/roundtrip.c) is compiled against include/fdtd.h,
linked with libfdtd_b200.so and — on a GPU box — run through create -> set_workspace -> forward -> reverse -> store_bytes;
its gradient is compared with the oracle's.  The CPU part checks that both headers are valid C99 on their own and that the
program links against every symbol it uses."""
import os
import struct
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
INC = os.path.join(ROOT, "include")
SRC = os.path.join(ROOT, "tests", "abi_c", "roundtrip.c")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")
GCC = ["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", f"-I{INC}", "-isystem", os.path.join(CUDA, "include")]


def _build_exe(tmp_path):
    from paper_2603_24027_b200 import build
    lib = build.build()
    exe = str(tmp_path / "roundtrip")
    libdir = os.path.dirname(lib)
    cmd = GCC + [SRC, "-o", exe, f"-L{libdir}", "-l:libfdtd_b200.so", f"-L{CUDA}/lib64", "-lcudart",
                 f"-Wl,-rpath,{libdir}", f"-Wl,-rpath,{CUDA}/lib64"]
    subprocess.check_call(cmd)
    return exe


@pytest.mark.parametrize("header", ["fdtd.h", "fdtd_bench.h"])
def test_headers_are_plain_c99(tmp_path, header):
    tu = tmp_path / "tu.c"
    tu.write_text(f'#include "{header}"\nint main(void) {{ return (int)FDTD_OK; }}\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", f"-I{INC}", "-fsyntax-only", str(tu)])


def test_c_program_compiles_and_links_against_the_library(tmp_path):
    exe = _build_exe(tmp_path)
    assert os.path.exists(exe)
    # without an input file it prints its usage and returns 1: the loader resolved libfdtd_b200.so and libcudart
    r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 1 and "usage" in r.stderr


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,k,interp", [(0, 1, 0), (2, 4, 0), (3, 5, 1)])
def test_c_program_round_trip_matches_the_oracle(tmp_path, dtype, k, interp):
    from oracle import fdtd_oracle as orc
    from paper_2603_24027_b200 import workloads as W
    exe = _build_exe(tmp_path)
    rng = np.random.default_rng(11)
    shape, P, T = (14, 13, 12), 3, 23
    eps = rng.uniform(1.0, 12.25, shape).astype(np.float32)
    src_comp, slo, shi = 2, (6, 6, 5), (8, 7, 7)
    wave = W.gauss_sine(T, 8, 3).astype(np.float32)
    dlo, dhi = (P, P, P), (shape[0] - P, shape[1] - P - 1, shape[2] - P)      # touches face, edge and corner shell cells
    clo, chi, cmask = (P + 1, P, P + 1), (P + 4, shape[1] - P, P + 5), 0b010101   # Ex, Ez, Hy
    ncomp = 3
    box = tuple(chi[a] - clo[a] for a in range(3))
    g = rng.standard_normal((ncomp,) + box).astype(np.float32)
    inp, out = tmp_path / "in.bin", tmp_path / "out.bin"
    with open(inp, "wb") as f:
        f.write(struct.pack("<8i", *shape, P, T, k, dtype, interp))
        f.write(struct.pack("<i3i3i", src_comp, *slo, *shi))
        f.write(struct.pack("<3i3i", *dlo, *dhi))
        f.write(struct.pack("<3i3iI", *clo, *chi, cmask))
        f.write(eps.tobytes())
        f.write(wave.tobytes())
        f.write(g.tobytes())
    r = subprocess.run([exe, str(inp), str(out)], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr + r.stdout
    raw = open(out, "rb").read()
    store_bytes = struct.unpack("<Q", raw[:8])[0]
    dshape = tuple(dhi[a] - dlo[a] for a in range(3))
    grad = np.frombuffer(raw[8:], dtype=np.float32).reshape(dshape).astype(np.float64)
    o = orc.OracleSim(32, eps, P, W.S)
    o.set_design(dlo, dhi)
    o.add_source(src_comp, slo, shi, None, wave)
    o.forward(T, dtype, k)
    dfinal = np.zeros((6,) + shape)
    for ci, comp in enumerate([c for c in range(6) if cmask >> c & 1]):
        dfinal[comp, clo[0]:chi[0], clo[1]:chi[1], clo[2]:chi[2]] = g[ci]
    og = o.reverse(dfinal, None, interp)
    assert np.abs(og).max() > 0
    err = np.linalg.norm(grad - og) / np.linalg.norm(og)
    print(f"[abi_c] dtype {dtype} k {k} interp {interp}: grad rel-L2 {err:.3e}, store {store_bytes} B")
    assert err <= 1e-4
    assert store_bytes == o.store_bytes()
