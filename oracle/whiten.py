"""Oracle injection + whitening ("We then inject the signals into the background
chunks ... We whiten the batch using the estimated power spectra").  DESIGN.md readings
R-I1..R-I7.  fp64.
"""
import numpy as np

from .fft import rfft, irfft


def psd_on_segment_grid(psd, n):
    """R-I4: linear interpolation of S (not sqrt S) from the Welch grid (n_psd bins, 0..Nyquist) to the
    segment grid (n/2+1 bins).  r = (n/2)/(n_psd-1) is an integer; bin j lies between Welch bins
    i0 = min(j // r, n_psd - 2) and i0 + 1 with weight t = (j - i0 r)/r."""
    psd = np.asarray(psd, dtype=np.float64)
    n_psd = psd.shape[-1]
    k = n // 2 + 1
    if n_psd == k:
        return psd.copy()
    r = (n // 2) // (n_psd - 1)
    assert r * (n_psd - 1) == n // 2
    j = np.arange(k)
    i0 = np.minimum(j // r, n_psd - 2)
    t = (j - i0 * r) / r
    return (1.0 - t) * psd[..., i0] + t * psd[..., i0 + 1]


def whitening_filter(psd, n, fs, f_lo, f_hi):
    """R-I2/R-I5: w[k] = sqrt(2 / (fs * S[k])) for f_lo <= f_k <= f_hi (inclusive), 0 elsewhere
    (the mask replaces the division outside the band, so S = 0 there is harmless)."""
    s = psd_on_segment_grid(psd, n)
    f = np.arange(n // 2 + 1) * (fs / n)
    band = (f >= f_lo) & (f <= f_hi)
    w = np.zeros_like(s)
    w[..., band] = np.sqrt(2.0 / (fs * s[..., band]))
    return w


def inject_whiten(noise, h_det, psd, fs, f_lo, f_hi):
    """out[b,d,:] = irfft( (rfft(noise[b,d,:]) + fs * h_det[b,d,:]) * w_d ).

    noise [B, D, N] real; h_det [B, D, K] complex or None (whiten only); psd [D, n_psd] in strain^2/Hz.
    R-I1: the signal is added in the frequency domain, X <- X + fs * h_d, which is the circular
    inverse DFT of h_d added in the time domain.  R-I7: all N samples are returned, no crop.
    """
    noise = np.asarray(noise, dtype=np.float64)
    n = noise.shape[-1]
    w = whitening_filter(psd, n, fs, f_lo, f_hi)              # [D, K]
    xk = rfft(noise)
    if h_det is not None:
        xk = xk + fs * np.asarray(h_det, dtype=np.complex128)
    return irfft(xk * w[None, :, :], n)


def gather(strip, offsets, n):
    """noise[b, d, :] = strip[d, offsets[b, d] : offsets[b, d] + n]  ("lazily loaded")."""
    strip = np.asarray(strip)
    offsets = np.asarray(offsets)
    b, d = offsets.shape
    out = np.empty((b, d, n), dtype=np.float64)
    for i in range(b):
        for j in range(d):
            o = int(offsets[i, j])
            out[i, j] = strip[j, o: o + n]
    return out


def optimal_snr(h_det, psd, n, fs, f_lo, f_hi):
    """Network optimal SNR rho = sqrt(sum_d 4 df sum_k |h_d|^2 / S_d) over the band (config c3)."""
    s = psd_on_segment_grid(psd, n)
    f = np.arange(n // 2 + 1) * (fs / n)
    band = (f >= f_lo) & (f <= f_hi)
    h_det = np.asarray(h_det)
    rho2 = 4.0 * (fs / n) * np.sum(np.abs(h_det[..., band]) ** 2 / s[..., band], axis=(-1, -2))
    return np.sqrt(rho2)
