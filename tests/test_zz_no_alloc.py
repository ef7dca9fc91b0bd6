"""amplfi_psd_welch_noalloc: the Welch estimate without a plan and without any device allocation (static scratch array).

Collected last on purpose (the suite runs with pytest -x).  Checked against the existing path, amplfi_psd_welch with a
plan, on two calls in a row that use the shared scratch array differently (the second must not see what the first left).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

if not torch.cuda.is_available():
    pytest.skip("needs a CUDA device", allow_module_level=True)

import paper_2407_19048_b200 as A          # noqa: E402  (fails loudly if libamplfi.so is missing)
import workloads as WL                     # noqa: E402

TOL = 1e-4                                 # PSD tolerance of tests/test_gpu_parity.py
DEV = "cuda:0"


def rel_err(got, ref, fs, nperseg):
    f = np.arange(nperseg // 2 + 1) * fs / nperseg
    band = (f >= 20.0) & (f <= 1000.0)
    g = got.cpu().numpy().astype(np.float64)[:, band]
    r = ref.cpu().numpy().astype(np.float64)[:, band]
    return np.abs(g / r - 1.0).max()


def test_noalloc_welch_matches_plan_path_on_two_calls_in_a_row():
    fs = 2048.0
    rng = np.random.Generator(np.random.Philox(0xA3D300AA))
    bg_a = torch.from_numpy(WL.coloured_noise(rng, (3,), 1 << 17, fs)).to(DEV)                 # 64 s: 63 segments of 4096
    strip = torch.from_numpy(WL.coloured_noise(rng, (2,), 1 << 18, fs) * np.float32(3.0)).to(DEV)
    bg_b = strip[:, 4097:4097 + 40000]             # a window of a strip (row stride > n_bg, odd start): 8 segments of 8192

    # existing path (plan-owned workspace)
    ref_a = A.amplfi_psd_welch(A.Plan(4096, fs, [0, 1, 2], 1, nperseg=4096), bg_a)
    ref_b = A.amplfi_psd_welch(A.Plan(8192, fs, [0, 1], 1, nperseg=8192), bg_b, detrend=0)

    # new entry point: outputs allocated up front, then two calls back to back with nothing in between
    out_a = torch.full((3, 2049), float("nan"), dtype=torch.float32, device=DEV)
    out_b = torch.full((2, 4097), float("nan"), dtype=torch.float32, device=DEV)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    A.amplfi_psd_welch_noalloc(bg_a, fs, 4096, out_a)
    A.amplfi_psd_welch_noalloc(bg_b, fs, 8192, out_b, detrend=0)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    assert bool(torch.isfinite(out_a).all()) and bool(torch.isfinite(out_b).all())
    assert rel_err(out_a, ref_a, fs, 4096) <= TOL
    assert rel_err(out_b, ref_b, fs, 8192) <= TOL

    # and the first shape again, after the array was used for the other one
    out_a2 = torch.full_like(out_a, float("nan"))
    A.amplfi_psd_welch_noalloc(bg_a, fs, 4096, out_a2)
    torch.cuda.synchronize()
    assert rel_err(out_a2, ref_a, fs, 4096) <= TOL
    assert torch.equal(out_a2, out_a)              # deterministic


def test_noalloc_welch_rejects_sizes_beyond_the_static_array():
    fs = 2048.0
    nperseg = 4096
    # 3 detectors x 255 segments x 2049 bins = 1.57 M floats > 2^20
    n_bg = nperseg + 254 * (nperseg // 2)
    bg = torch.zeros((3, n_bg), dtype=torch.float32, device=DEV)
    out = torch.full((3, nperseg // 2 + 1), 7.0, dtype=torch.float32, device=DEV)
    assert 3 * 255 * (nperseg // 2 + 1) > A.NOALLOC_WELCH_FLOATS
    with pytest.raises(A.AmplfiError) as err:
        A.amplfi_psd_welch_noalloc(bg, fs, nperseg, out)
    assert "static array" in str(err.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                # nothing was launched
    with pytest.raises(A.AmplfiError):
        A.amplfi_psd_welch_noalloc(bg, fs, 3000, out)          # not a power of two
