"""Oracle Welch power-spectrum estimate ("power spectra estimation",
PAPER.md:103 "The power spectra is fit to this background chunk").  The estimator is not
named in the paper; BASELINE.json's configs fix Welch / Hann / 50 % overlap / mean.
DESIGN.md readings R-S1..R-S6.  fp64.
"""
import numpy as np

from .fft import rfft


def hann_periodic(nperseg):
    """R-S2: w[n] = (1 - cos(2 pi n / nperseg)) / 2."""
    return 0.5 * (1.0 - np.cos(2.0 * np.pi * np.arange(nperseg) / nperseg))


def welch(x, fs, nperseg, noverlap=None, detrend=1):
    """One-sided density S[k], k = 0..nperseg/2, of the real sequence(s) x[..., n_bg].

    R-S1: segments start at j*step, step = nperseg - noverlap, full segments only.
    R-S3: detrend=1 subtracts each segment's mean before the window; 0 does nothing.
    R-S4: S[k] = c_k * mean_j |FFT(w * x_j)[k]|^2 / (fs * sum w^2), c_k = 2 except DC and Nyquist (1).
    R-S5: plain mean over segments.
    """
    x = np.asarray(x, dtype=np.float64)
    if noverlap is None:
        noverlap = nperseg // 2
    step = nperseg - noverlap
    n_bg = x.shape[-1]
    nseg = (n_bg - nperseg) // step + 1
    w = hann_periodic(nperseg)
    acc = np.zeros(x.shape[:-1] + (nperseg // 2 + 1,))
    for j in range(nseg):
        seg = x[..., j * step: j * step + nperseg]
        if detrend:
            seg = seg - seg.mean(axis=-1, keepdims=True)
        acc += np.abs(rfft(seg * w)) ** 2
    psd = acc / nseg / (fs * np.sum(w * w))
    psd[..., 1:-1] *= 2.0
    return psd
