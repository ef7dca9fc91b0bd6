"""Pins for oracle.fft (BASELINE north_star check "Parseval")."""
import numpy as np
import pytest

from oracle import fft as F


@pytest.mark.parametrize("n", [2, 8, 64, 128, 1024, 4096])
def test_matches_numpy(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal((3, n)) + 1j * rng.standard_normal((3, n))
    ref = np.fft.fft(x)
    assert np.abs(F.fft(x) - ref).max() <= 1e-12 * np.abs(ref).max()
    assert np.abs(F.ifft(x) - np.fft.ifft(x)).max() <= 1e-12
    xr = x.real
    assert np.abs(F.rfft(xr) - np.fft.rfft(xr)).max() <= 1e-12 * np.abs(ref).max()
    spec = np.fft.rfft(xr)
    assert np.abs(F.irfft(spec, n) - np.fft.irfft(spec, n)).max() <= 1e-12


def test_naive_equals_recursive():
    rng = np.random.default_rng(1)
    x = rng.standard_normal(256) + 1j * rng.standard_normal(256)
    assert np.abs(F.dft_naive(x) - F.fft_recursive(x)).max() < 1e-11


def test_sign_convention_single_tone():
    # x[n] = exp(+2 pi i 3 n / N) must land in bin +3 of the FORWARD transform (kernel e^{-i...})
    n = 128
    x = np.exp(2j * np.pi * 3 * np.arange(n) / n)
    xk = F.fft(x)
    assert abs(xk[3] - n) < 1e-9 and np.abs(np.delete(xk, 3)).max() < 1e-9


def test_impulse_flat_and_shift():
    n = 256
    x = np.zeros(n)
    x[5] = 1.0
    xk = F.rfft(x)
    k = np.arange(n // 2 + 1)
    assert np.abs(xk - np.exp(-2j * np.pi * k * 5 / n)).max() < 1e-12


@pytest.mark.parametrize("n", [16, 64, 2048])
def test_parseval(n):
    x = np.random.default_rng(7).standard_normal(n)
    xk = F.rfft(x)
    lhs = np.sum(x * x)
    rhs = (abs(xk[0]) ** 2 + 2 * np.sum(np.abs(xk[1:-1]) ** 2) + abs(xk[-1]) ** 2) / n
    assert abs(lhs - rhs) <= 1e-12 * lhs


def test_irfft_ignores_dc_nyquist_imag():
    n = 64
    spec = np.fft.rfft(np.random.default_rng(3).standard_normal(n))
    spec2 = spec.copy()
    spec2[0] += 5j
    spec2[-1] -= 2j
    assert np.abs(F.irfft(spec2, n) - F.irfft(spec, n)).max() < 1e-14
