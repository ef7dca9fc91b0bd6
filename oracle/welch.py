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


def median_bias(nseg):
    """Ratio E[median]/E[mean] of nseg independent periodogram values (each exponentially distributed, i.e.
    chi-squared with 2 degrees of freedom).  The k-th smallest of n unit exponentials has expectation
    sum_{j=n-k+1}^{n} 1/j; the median is the middle order statistic (odd n) or the mean of the two middle ones
    (even n, numpy.median's convention).  For odd n this equals the alternating harmonic sum
    1 - 1/2 + 1/3 - ... + 1/n (-> ln 2)."""
    def e_order(k):
        return sum(1.0 / j for j in range(nseg - k + 1, nseg + 1))
    if nseg % 2:
        return e_order((nseg + 1) // 2)
    return 0.5 * (e_order(nseg // 2) + e_order(nseg // 2 + 1))


def welch(x, fs, nperseg, noverlap=None, detrend=1, average="mean"):
    """One-sided density S[k], k = 0..nperseg/2, of the real sequence(s) x[..., n_bg].

    R-S1: segments start at j*step, step = nperseg - noverlap, full segments only.
    R-S3: detrend=1 subtracts each segment's mean before the window; 0 does nothing.
    R-S4: S[k] = c_k * mean_j |FFT(w * x_j)[k]|^2 / (fs * sum w^2), c_k = 2 except DC and Nyquist (1).
    R-S5: plain mean over segments; average="median" takes, per bin, the median over
          segments divided by median_bias(nseg), which is robust against loud transients in the background.
    """
    x = np.asarray(x, dtype=np.float64)
    if noverlap is None:
        noverlap = nperseg // 2
    step = nperseg - noverlap
    n_bg = x.shape[-1]
    nseg = (n_bg - nperseg) // step + 1
    w = hann_periodic(nperseg)
    per = np.zeros((nseg,) + x.shape[:-1] + (nperseg // 2 + 1,))
    for j in range(nseg):
        seg = x[..., j * step: j * step + nperseg]
        if detrend:
            seg = seg - seg.mean(axis=-1, keepdims=True)
        per[j] = np.abs(rfft(seg * w)) ** 2
    if average == "mean":
        acc = np.zeros(per.shape[1:])
        for j in range(nseg):
            acc += per[j]
        avg = acc / nseg
    elif average == "median":
        avg = np.median(per, axis=0) / median_bias(nseg)
    else:
        raise ValueError(average)
    psd = avg / (fs * np.sum(w * w))
    psd[..., 1:-1] *= 2.0
    return psd
