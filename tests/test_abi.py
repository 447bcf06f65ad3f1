"""The C-ABI library loads and exports every symbol include/et.h declares (no compute without a GPU)."""
import ctypes
import os
import re

import pytest

from paper_1612_04705_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def header_functions():
    src = open(os.path.join(ROOT, "include", "et.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(et_[a-zA-Z_]+)\s*\(", src)))


def test_header_and_binding_list_the_same_symbols():
    assert header_functions() == sorted(binding.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in header_functions():
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.et_version()


def test_no_cpu_fallback(lib):
    """Without a CUDA device et_create must fail loudly (ET_ERR_CUDA), never compute on the CPU."""
    try:
        import torch

        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        pytest.skip("a GPU is present")
    h = ctypes.c_void_p()
    assert lib.et_create(ctypes.byref(h), 0, None) == -6
    with pytest.raises(binding.EtError):
        binding.Context(0)


def test_product_does_not_import_oracle():
    """The product path may not route through the oracle."""
    pkg = os.path.join(ROOT, "paper_1612_04705_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "et_oracle" not in text, f


def test_struct_sizes_match_header(lib):
    # et_result: 9 doubles + int64; et_perm_result adds double + 3 int64; et_stats 3 doubles + 2 int64
    assert ctypes.sizeof(binding._Result) == 80
    assert ctypes.sizeof(binding._PermResult) == 80 + 32
    assert ctypes.sizeof(binding._PoddResult) == 32 + 80 + 112
    assert ctypes.sizeof(binding._Stats) == 40 + 24 + 32 + 5 * 8
    assert ctypes.sizeof(binding._BkgResult) == 4 * 8 + 10 * 8 + 2 * 8 + 8
    assert ctypes.sizeof(binding._BkgPermResult) == (4 + 10 + 2 + 1) * 8 + 4 * 8
    assert ctypes.sizeof(binding._GevResult) == 3 * 8 + 9 * 8 + 5 * 8 + 3 * 8
    assert ctypes.sizeof(binding._ScpResult) == 9 * 8


C_CALLER = os.path.join(ROOT, "tests", "c_caller.c")


def build_c_caller(tmp_path):
    """tests/c_caller.c is a plain C program that includes include/et.h and links libet.so: the boundary is a C ABI."""
    import subprocess

    exe = str(tmp_path / "c_caller")
    libdir = os.path.dirname(binding.LIB_PATH)
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-I", os.path.join(ROOT, "include"), C_CALLER, "-o", exe,
                           "-L", libdir, "-l:libet.so", "-Wl,-rpath," + libdir, "-lm"])
    return exe


def test_c_caller_compiles_and_fails_loudly_without_a_gpu(lib, tmp_path):
    import subprocess

    try:
        import torch

        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    exe = build_c_caller(tmp_path)
    r = subprocess.run([exe], capture_output=True, text=True)
    if has_gpu:
        assert r.returncode == 0 and "T = 0.125" in r.stdout, r.stdout + r.stderr
    else:
        assert r.returncode == 3 and "et_create failed: -6" in r.stdout, r.stdout + r.stderr


@pytest.mark.gpu
def test_c_caller_runs_et_T_on_the_gpu(lib, tmp_path):
    """Pin P2 (2 + 2 square, T = 0.125) and a 3000-event et_T / et_permutation_test from a C program: no Python between
    the caller and the library."""
    import subprocess

    r = subprocess.run([build_c_caller(tmp_path)], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "T = 0.125" in r.stdout and "permutation test ok" in r.stdout, r.stdout


def test_static_entry_point_fails_loudly_without_setup_or_device(lib):
    """et_T_static (the entry point that allocates nothing) never computes without its set-up: without a CUDA device
    et_static_setup reports ET_ERR_CUDA, and a call on a device that was not set up is ET_ERR_INVALID with a message."""
    try:
        import torch

        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if not has_gpu:
        assert lib.et_static_setup(0) == -6
        assert b"CUDA" in lib.et_static_last_error()
    buf = (ctypes.c_double * 16)()
    out = (ctypes.c_double * 10)()
    p = ctypes.cast(buf, ctypes.c_void_p)
    st = lib.et_T_static(63, None, p, 4, p, 4, 2, 1, 0.3, ctypes.cast(out, ctypes.c_void_p))  # device 63 is never set up
    assert st == -1 and b"et_static_setup" in lib.et_static_last_error()
    assert lib.et_T_static(63, None, None, 4, p, 4, 2, 1, 0.3, ctypes.cast(out, ctypes.c_void_p)) == -1
    assert lib.et_T_static(63, None, p, 4, p, 4, 2, 1, -1.0, ctypes.cast(out, ctypes.c_void_p)) == -2
