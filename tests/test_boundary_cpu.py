"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, loads without a GPU, and exports
every symbol include/pfsm.h declares.  No compute calls here."""
import ctypes
import os
import re

import pytest

import paper_1502_07806_b200 as pfsm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "pfsm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pfsm_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_three_core_calls():
    syms = declared_symbols()
    for core in ("pfsm_create", "pfsm_solve", "pfsm_destroy"):
        assert core in syms


def test_library_loads_and_exports_every_declared_symbol():
    lib = pfsm.load()
    syms = declared_symbols()
    assert sorted(syms) == sorted(pfsm.EXPORTS)
    for name in syms:
        assert hasattr(lib, name), name


def test_library_is_sm100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", pfsm.lib_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(7|8|9)\d", out)


def test_strerror_and_null_handle_paths():
    lib = pfsm.load()
    assert pfsm.strerror(0) == "success"
    assert "argument 3" in pfsm.strerror(-3)
    assert lib.pfsm_destroy(None) == 0
    assert lib.pfsm_solve(None, None, None, None, None) == -1
    assert lib.pfsm_workspace_bytes(None) == 0


def test_create_rejects_bad_arguments_before_touching_cuda():
    lib = pfsm.load()
    h = ctypes.c_void_p()
    assert lib.pfsm_create(None, 256, 4, 16, 3, 0.5) == -1
    assert lib.pfsm_create(ctypes.byref(h), 1, 1, 0, 1, 0.5) == -2      # N < 2
    assert lib.pfsm_create(ctypes.byref(h), 256, 0, 16, 3, 0.5) == -3   # P < 1
    assert lib.pfsm_create(ctypes.byref(h), 256, 257, 0, 3, 0.5) == -3  # P > N would leave a slice empty (reading R14)
    assert lib.pfsm_create(ctypes.byref(h), 256, 4, -1, 3, 0.5) == -4
    assert lib.pfsm_create(ctypes.byref(h), 32768, 2, 0, 3, 0.5) == -4  # M = 16384 > 8192 unsupported in this version
    assert lib.pfsm_create(ctypes.byref(h), 256, 4, 16, -1, 0.5) == -5
    assert lib.pfsm_create(ctypes.byref(h), 256, 4, 16, 3, 0.0) == -6
    assert lib.pfsm_create(ctypes.byref(h), 256, 4, 16, 3, float("nan")) == -6
    assert not h.value


def test_no_gpu_means_loud_failure_not_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        pfsm.Handle(256, 4, 16, 3, 0.5)
    # and the raw C call reports a CUDA error code, not success
    h = ctypes.c_void_p()
    rc = pfsm.load().pfsm_create(ctypes.byref(h), 256, 4, 16, 3, 0.5)
    assert rc >= pfsm.CUDA_ERROR_BASE
