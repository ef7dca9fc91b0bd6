"""Oracle Fourier transforms ("fourier transforms ... are carried out on the GPU").

Definition followed (reading R-W4): forward X[k] = sum_n x[n] exp(-2 pi i k n / N),
inverse x[n] = (1/N) sum_k X[k] exp(+2 pi i k n / N).  A naive O(N^2) DFT is used for
N <= 64 and a plain recursive radix-2 decimation-in-time FFT above that (BASELINE.json
north_star).  All transforms act on the last axis; leading axes are batch.
"""
import numpy as np

NAIVE_MAX = 64


def dft_naive(x, sign=-1):
    """X[k] = sum_n x[n] exp(sign * 2 pi i k n / N), written out as a matrix product."""
    x = np.asarray(x, dtype=np.complex128)
    n = x.shape[-1]
    idx = np.arange(n)
    w = np.exp(sign * 2j * np.pi * np.outer(idx, idx) / n)     # w[k, n]
    return x @ w.T


def fft_recursive(x, sign=-1):
    """Radix-2 DIT recursion: X[k] = E[k] + w^k O[k], X[k+N/2] = E[k] - w^k O[k]."""
    x = np.asarray(x, dtype=np.complex128)
    n = x.shape[-1]
    if n <= NAIVE_MAX or n % 2:
        return dft_naive(x, sign)
    even = fft_recursive(x[..., 0::2], sign)
    odd = fft_recursive(x[..., 1::2], sign)
    w = np.exp(sign * 2j * np.pi * np.arange(n // 2) / n)
    return np.concatenate([even + w * odd, even - w * odd], axis=-1)


def fft(x):
    return fft_recursive(x, -1)


def ifft(x):
    x = np.asarray(x, dtype=np.complex128)
    return fft_recursive(x, +1) / x.shape[-1]


def rfft(x):
    """One-sided spectrum of a real sequence: bins 0 .. N/2."""
    x = np.asarray(x, dtype=np.float64)
    n = x.shape[-1]
    return fft_recursive(x.astype(np.complex128), -1)[..., : n // 2 + 1]


def irfft(xk, n):
    """Real sequence whose one-sided spectrum is xk (length n/2+1), n even.

    The full spectrum is rebuilt by Hermitian symmetry X[n-k] = conj(X[k]); the imaginary
    parts of the DC and Nyquist bins are dropped (they cannot belong to a real sequence).
    """
    xk = np.asarray(xk, dtype=np.complex128)
    assert n % 2 == 0 and xk.shape[-1] == n // 2 + 1
    full = np.empty(xk.shape[:-1] + (n,), dtype=np.complex128)
    full[..., : n // 2 + 1] = xk
    full[..., 0] = xk[..., 0].real
    full[..., n // 2] = xk[..., n // 2].real
    full[..., n // 2 + 1:] = np.conj(xk[..., 1: n // 2][..., ::-1])
    return (fft_recursive(full, +1) / n).real
