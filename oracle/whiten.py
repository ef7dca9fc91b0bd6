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


# ----------------------------------------------------------------------------------------
# whitening with a time-truncated filter (the practice of the library the paper
# delegates to; the paper itself prints nothing).  DESIGN.md reading R-I8.
# ----------------------------------------------------------------------------------------

def fir_truncated_filter(psd, n, fs, f_lo, f_hi, fduration):
    """Frequency response W'[k], k = 0..n/2, of the whitening filter truncated in time to fduration seconds.

    Step by step (R-I8):
      1. w[k] = sqrt(2 / (fs S[k])) inside [f_lo, f_hi], 0 outside      (whitening_filter above)
      2. q = irfft(w): the zero-phase impulse response, real and even, q[j] = q[n - j]
      3. taper to ntaps = fduration * fs samples around lag 0 with a Hann window centred on lag 0:
             q'[j] = q[j] * (1 + cos(2 pi m / ntaps)) / 2   for m = min(j, n - j) < ntaps / 2,   0 otherwise
      4. W' = rfft(q')   (real, because q' is even; the imaginary rounding residue is dropped)
    The response no longer vanishes exactly outside the band and no mask is re-applied.
    """
    w = whitening_filter(psd, n, fs, f_lo, f_hi)
    ntaps = int(round(fduration * fs))
    assert 2 <= ntaps <= n and ntaps % 2 == 0
    q = irfft(w.astype(np.complex128), n)
    j = np.arange(n)
    m = np.minimum(j, n - j)
    taper = np.where(m < ntaps // 2, 0.5 * (1.0 + np.cos(2.0 * np.pi * m / ntaps)), 0.0)
    return rfft(q * taper).real


def inject_whiten_fir(noise, h_det, psd, fs, f_lo, f_hi, fduration, crop=True):
    """out = irfft( (rfft(noise) + fs h_det) * W' ), W' = fir_truncated_filter; with crop the first and last
    fduration/2 seconds, which the circular convolution contaminates with samples from the other end of the
    segment, are removed: out has n - ntaps samples.  Inside the crop the result equals the LINEAR convolution
    of the data with the ntaps-long filter (pinned against numpy.convolve)."""
    noise = np.asarray(noise, dtype=np.float64)
    n = noise.shape[-1]
    wf = fir_truncated_filter(psd, n, fs, f_lo, f_hi, fduration)
    xk = rfft(noise)
    if h_det is not None:
        xk = xk + fs * np.asarray(h_det, dtype=np.complex128)
    y = irfft(xk * wf[None, :, :], n)
    if not crop:
        return y
    pad = int(round(fduration * fs)) // 2
    return y[..., pad: n - pad]
