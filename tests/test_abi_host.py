"""Host-side checks of the C-ABI library (no GPU needed): it builds, loads, exports every symbol that
include/amplfi.h declares, validates arguments before touching the device, and its IMRPhenomD fit table
equals the oracle's copy."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import __graft_entry__ as G      # noqa: E402


@pytest.fixture(scope="module")
def lib():
    G.build()                     # cross-compiles for sm_100a without a GPU
    import paper_2407_19048_b200 as A
    return A


def header_functions():
    text = open(os.path.join(ROOT, "include", "amplfi.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(amplfi_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    declared = header_functions()
    assert {"amplfi_waveform_fd", "amplfi_project", "amplfi_psd_welch", "amplfi_inject_whiten"} <= set(declared)
    raw = ctypes.CDLL(lib.LIB_PATH)
    for name in declared:
        assert hasattr(raw, name), "libamplfi.so does not export %s" % name
    assert set(declared) == set(lib.EXPORTS)
    # the symbols are plain C (no C++ mangling) and the kernels are sm_100a code
    nm = subprocess.run(["nm", "-D", "--defined-only", lib.LIB_PATH], capture_output=True, text=True).stdout
    for name in declared:
        assert re.search(r"\bT %s$" % name, nm, flags=re.M)


def test_sass_is_sm100a(lib):
    out = subprocess.run(["cuobjdump", "-lelf", lib.LIB_PATH], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump not available")
    assert "sm_100a" in out.stdout


def test_constants(lib):
    assert lib.psd_scale() == 2.0 ** 140
    assert "sm_100a" in lib.version()
    assert lib.launch_count() >= 0


def test_phenomd_table_matches_oracle_copy(lib):
    from oracle import phenomd_coeffs as T
    got = np.array(lib.phenomd_table())
    want = np.array([T.TABLE[name] for name in T.NAMES])
    assert got.shape == (19, 11)
    assert np.array_equal(got, want)


def test_kerr_mode_table_of_the_library_against_the_oracle_solver(lib):
    """The library tabulates the Kerr (2,2,0) mode with its own C++ continued-fraction solver (csrc/kerr_qnm.cu, host code:
    no GPU needed); the oracle's Python solver / table (oracle/qnm.py) is an independent implementation of Leaver's method."""
    from oracle import qnm
    spins, w_re, w_im = lib.qnm_table()
    assert len(spins) == 512 and abs(spins[0] - 0.998) < 1e-12 and abs(spins[-1] + 0.998) < 1e-12
    for i in range(0, 512, 7):
        r, im = qnm.qnm_220(spins[i])
        tol = 1e-8 if abs(spins[i]) <= 0.98 else 1e-6           # (the oracle's spline is coarser next to the extremal hole)
        assert abs(w_re[i] / r - 1.0) < tol and abs(w_im[i] / im - 1.0) < tol
    i0 = min(range(512), key=lambda i: abs(spins[i]))
    w, _ = qnm.kerr_qnm_220(spins[i0])                      # a direct solve, not the oracle's table
    assert abs(w_re[i0] - w.real) < 1e-10 and abs(w_im[i0] + w.imag) < 1e-10


def test_argument_validation_without_device(lib):
    L = lib._lib
    h = ctypes.c_void_p()
    ids = (ctypes.c_int * 3)(0, 1, 2)
    bad = (ctypes.c_int * 3)(0, 7, 2)
    # invalid arguments are rejected before any CUDA call
    assert L.amplfi_plan_create(8192, 2048.0, 3, ids, 4, 0, None) == lib.ERR_INVALID_ARG
    assert L.amplfi_plan_create(8192, 2048.0, 0, ids, 4, 0, ctypes.byref(h)) == lib.ERR_INVALID_ARG
    assert L.amplfi_plan_create(8192, 2048.0, 3, bad, 4, 0, ctypes.byref(h)) == lib.ERR_INVALID_ARG
    assert b"detector" in L.amplfi_last_error()
    assert L.amplfi_plan_create(8192, -1.0, 3, ids, 4, 0, ctypes.byref(h)) == lib.ERR_INVALID_ARG
    assert L.amplfi_plan_create(8192, 2048.0, 3, ids, 0, 0, ctypes.byref(h)) == lib.ERR_INVALID_ARG
    assert L.amplfi_plan_create(8000, 2048.0, 3, ids, 4, 0, ctypes.byref(h)) == lib.ERR_UNSUPPORTED_SIZE
    assert L.amplfi_plan_create(512, 2048.0, 3, ids, 4, 0, ctypes.byref(h)) == lib.ERR_UNSUPPORTED_SIZE
    assert L.amplfi_plan_create(1 << 21, 2048.0, 3, ids, 4, 0, ctypes.byref(h)) == lib.ERR_UNSUPPORTED_SIZE
    assert L.amplfi_plan_create(8192, 2048.0, 3, ids, 4, 3000, ctypes.byref(h)) == lib.ERR_UNSUPPORTED_SIZE
    assert h.value is None
    # null plan / null buffers
    assert L.amplfi_waveform_fd(None, 0, 1, None, 20.0, 1000.0, None, None, None, None) == lib.ERR_INVALID_ARG
    assert L.amplfi_project(None, 1, None, 0.0, None, None, None, None, None) == lib.ERR_INVALID_ARG
    assert L.amplfi_psd_welch(None, None, 0, 0, 0, 0, 0, None, None) == lib.ERR_INVALID_ARG
    assert L.amplfi_inject_whiten(None, 1, None, None, 0, None, 0, None, 0.0, None, 0, 20.0, 1000.0, None, None) \
        == lib.ERR_INVALID_ARG
    assert L.amplfi_phenomd_table(None) == lib.ERR_INVALID_ARG
    assert L.amplfi_plan_set_timing(None, 1) == lib.ERR_INVALID_ARG
    L.amplfi_plan_destroy(None)              # must be a no-op


def test_no_device_is_an_error_not_a_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(lib.AmplfiError) as ei:
        lib.Plan(8192, 2048.0, [0, 1], 4)
    assert ei.value.code == lib.ERR_CUDA
    fake = object.__new__(lib.Plan)
    fake.nperseg, fake.n_det, fake._h = 4096, 2, None
    with pytest.raises(TypeError):
        lib.amplfi_psd_welch(fake, torch.zeros(2, 8192))


def test_binding_rejects_cpu_tensors(lib):
    import torch

    class FakePlan:
        _h = None
        n, n_bins, n_det, nperseg = 8192, 4097, 2, 4096
    with pytest.raises(TypeError):
        lib.amplfi_waveform_fd(FakePlan(), 0, torch.zeros(2, 11, dtype=torch.float64), 20.0, 1000.0,
                               hp=torch.zeros(2, 4097, 2), hc=torch.zeros(2, 4097, 2), flags=torch.zeros(2, dtype=torch.int32))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2407_19048_b200")
    for base, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(base, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "_work" not in text, f
