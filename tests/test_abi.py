"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/rna4r.h declares; argument validation that needs no GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "rna4r.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rna4r_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1307_7820_b200 import build
    path = build.build()
    lib = ctypes.CDLL(path)
    names = declared_symbols()
    assert len(names) >= 15
    for nm in names:
        assert hasattr(lib, nm), nm


def test_header_compiles_as_c_and_a_c_program_calls_the_abi(tmp_path):
    """include/rna4r.h is a C header: a C99 program includes it, links librna4r.so and calls the GPU-free entry points."""
    import subprocess
    from paper_1307_7820_b200 import build
    lib = build.build()
    exe = str(tmp_path / "c_abi_check")
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                           os.path.join(ROOT, "tests", "c_abi_check.c"), "-o", exe,
                           "-L", os.path.dirname(lib), "-lrna4r", "-Wl,-rpath," + os.path.dirname(lib)])
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0, (out.returncode, out.stdout, out.stderr)
    assert "c_abi_check ok" in out.stdout


def test_smem_engine_layout_fits_config4(tmp_path):
    """the SMEM engine's shared-memory plan (host logic): config 4's longest sequence fits, regions aligned and disjoint"""
    import shutil
    import subprocess
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc not on PATH")
    exe = str(tmp_path / "smem_layout_check")
    subprocess.check_call(["nvcc", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe,
                           os.path.join(ROOT, "tests", "smem_layout_check.cu")])
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0, (out.returncode, out.stdout)
    assert "smem_layout_check ok" in out.stdout and "q=8 max_n=70" in out.stdout


def test_strerror_and_version_need_no_gpu():
    from paper_1307_7820_b200 import load
    L = load()
    assert L.rna4r_version().decode().startswith("rna4r")
    assert L.rna4r_strerror(0).decode() == "ok"
    for code in range(-10, 0):
        assert len(L.rna4r_strerror(code).decode()) > 3


def test_prepare_rejects_bad_q_and_null_before_touching_cuda():
    from paper_1307_7820_b200 import load
    L = load()
    h = ctypes.c_void_p()
    assert L.rna4r_prepare(1, 0, None, ctypes.byref(h)) == -1
    assert L.rna4r_prepare(13, 0, None, ctypes.byref(h)) == -1
    assert L.rna4r_prepare(8, 0, None, None) == -2
    assert L.rna4r_destroy(None) == -5
    assert L.rna4r_workspace_bytes(None, 10, 1, 0) == 0


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1307_7820_b200 import load, Rna4r
    h = ctypes.c_void_p()
    assert load().rna4r_prepare(8, 0, None, ctypes.byref(h)) == -7   # RNA4R_ERR_DEVICE
    with pytest.raises(RuntimeError):
        Rna4r(8)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1307_7820_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
