"""Pins for oracle.welch and oracle.whiten (BASELINE north_star checks
"linearity of injection", "whitened pure Gaussian noise having unit variance per bin")."""
import numpy as np
import pytest
import scipy.signal

from oracle import fft as F
from oracle import welch as WE
from oracle import whiten as WH
from workloads import aligo_psd, coloured_noise

from conftest import read_golden


@pytest.mark.parametrize("detrend", [0, 1])
@pytest.mark.parametrize("n_bg,nperseg", [(4096, 256), (5000, 512), (131072, 4096)])
def test_welch_matches_scipy(n_bg, nperseg, detrend):
    # S-4: scipy pins the ORACLE (the GPU is compared with the oracle, never with scipy)
    x = np.random.default_rng(n_bg).standard_normal((2, n_bg)) * 3.0 + 0.7
    got = WE.welch(x, 2048.0, nperseg, detrend=detrend)
    _, ref = scipy.signal.welch(x, 2048.0, "hann", nperseg, nperseg // 2,
                                detrend="constant" if detrend else False, scaling="density", average="mean")
    assert np.abs(got - ref).max() <= 1e-12 * ref.max()


def test_welch_segment_count_and_window():
    # S-1: 63 segments in every BASELINE config; S-2: periodic Hann
    for n_bg, nps in ((131072, 4096), (262144, 8192), (524288, 16384)):
        assert (n_bg - nps) // (nps // 2) + 1 == 63
    assert np.allclose(WE.hann_periodic(8), scipy.signal.get_window("hann", 8, fftbins=True))
    assert WE.hann_periodic(8)[0] == 0 and abs(WE.hann_periodic(8)[4] - 1) < 1e-15


def test_welch_white_noise_level_and_parseval():
    # white noise of variance s^2 sampled at fs has one-sided density 2 s^2 / fs
    fs, s = 2048.0, 3.0
    x = np.random.default_rng(0).standard_normal(1 << 18) * s
    psd = WE.welch(x, fs, 1024, detrend=0)
    assert abs(psd[5:-5].mean() / (2 * s * s / fs) - 1) < 0.01
    assert abs(psd.sum() * fs / 1024 / (s * s) - 1) < 0.02          # integral of S df = variance


def test_welch_recovers_coloured_psd():
    # S-7: mean(S_hat / S_true) = 1 in band
    fs, n = 2048.0, 1 << 19
    x = coloured_noise(np.random.Generator(np.random.Philox(11)), (1,), n, fs, dtype=np.float64)[0]
    psd = WE.welch(x, fs, 4096)
    f = np.arange(2049) * fs / 4096
    band = (f >= 40) & (f <= 900)
    assert abs(np.mean(psd[band] / aligo_psd(f[band])) - 1) < 0.01


def test_aligo_psd_golden():
    g = read_golden("aligo_psd_values.txt")
    assert abs(aligo_psd(215.0) / 3.3e-48 - 1) < 1e-12
    assert np.abs(aligo_psd(np.array(g["f"])) / np.array(g["S"]) - 1).max() < 1e-4
    assert aligo_psd(5.0) == aligo_psd(20.0)


@pytest.mark.parametrize("n,n_psd", [(64, 17), (64, 9), (16384, 2049), (65536, 8193), (256, 129)])
def test_psd_interp_equals_numpy_interp(n, n_psd):
    s = np.random.default_rng(n).uniform(1, 2, (3, n_psd))
    got = WH.psd_on_segment_grid(s, n)
    fk = np.arange(n // 2 + 1) / n
    fw = np.arange(n_psd) / (2.0 * (n_psd - 1))
    for d in range(3):
        assert np.abs(got[d] - np.interp(fk, fw, s[d])).max() < 1e-14
    assert got.shape == (3, n // 2 + 1)


def test_whiten_brute_force_tiny():
    # I-2/I-5 written out with explicit DFT matrices on N = 32, band edges inclusive
    n, fs, f_lo, f_hi = 32, 64.0, 6.0, 20.0
    rng = np.random.default_rng(4)
    x = rng.standard_normal((2, 1, n))
    h = rng.standard_normal((2, 1, n // 2 + 1)) + 1j * rng.standard_normal((2, 1, n // 2 + 1))
    s = rng.uniform(0.5, 2.0, (1, n // 2 + 1))
    got = WH.inject_whiten(x, h, s, fs, f_lo, f_hi)
    idx = np.arange(n)
    fwd = np.exp(-2j * np.pi * np.outer(idx, idx) / n)
    for b in range(2):
        full = fwd @ x[b, 0]
        out = np.zeros(n)
        for k in range(n // 2 + 1):
            fk = k * fs / n
            if fk < f_lo or fk > f_hi:
                continue
            val = (full[k] + fs * h[b, 0, k]) * np.sqrt(2.0 / (fs * s[0, k]))
            wgt = 1.0 if k in (0, n // 2) else 2.0
            out += wgt * (val * np.exp(2j * np.pi * k * idx / n)).real / n
        assert np.abs(out - got[b, 0]).max() < 1e-12
    assert 6.0 == 3 * fs / n and 20.0 == 10 * fs / n         # both edges sit exactly on bins (inclusive)


def test_injection_is_linear():
    # north_star check: whiten(n + a h1 + b h2) = whiten(n) + a whiten(h1) + b whiten(h2)
    n, fs = 1024, 2048.0
    rng = np.random.default_rng(8)
    x = rng.standard_normal((1, 2, n)) * 1e-21
    k = n // 2 + 1
    h1 = (rng.standard_normal((1, 2, k)) + 1j * rng.standard_normal((1, 2, k))) * 1e-24
    h2 = (rng.standard_normal((1, 2, k)) + 1j * rng.standard_normal((1, 2, k))) * 1e-24
    s = np.tile(aligo_psd(np.arange(k) * fs / n), (2, 1))
    zero = np.zeros_like(x)
    a, b = 0.7, -2.5
    lhs = WH.inject_whiten(x, a * h1 + b * h2, s, fs, 20.0, 1000.0)
    rhs = (WH.inject_whiten(x, None, s, fs, 20.0, 1000.0) + a * WH.inject_whiten(zero, h1, s, fs, 20.0, 1000.0)
           + b * WH.inject_whiten(zero, h2, s, fs, 20.0, 1000.0))
    assert np.abs(lhs - rhs).max() < 1e-12 * np.abs(lhs).max()


def test_fd_injection_equals_time_domain_addition():
    # I-1: X + fs h  ==  rfft(x + irfft(fs h))
    n, fs = 512, 2048.0
    rng = np.random.default_rng(12)
    x = rng.standard_normal((1, 1, n))
    k = n // 2 + 1
    h = rng.standard_normal((1, 1, k)) + 1j * rng.standard_normal((1, 1, k))
    h[..., 0] = 0
    h[..., -1] = 0
    s = np.ones((1, k))
    a = WH.inject_whiten(x, h, s, fs, 20.0, 1000.0)
    b = WH.inject_whiten(x + F.irfft(fs * h, n), None, s, fs, 20.0, 1000.0)
    assert np.abs(a - b).max() < 1e-11


def test_whitened_gaussian_noise_has_unit_variance_per_bin():
    # I-2: periodic Gaussian noise with one-sided PSD S: E|W[k]|^2 / N = 1; time-domain variance = kept-band fraction
    fs, n, reps = 2048.0, 4096, 200
    x = coloured_noise(np.random.Generator(np.random.Philox(21)), (reps, 1), n, fs, dtype=np.float64)
    k = n // 2 + 1
    f = np.arange(k) * fs / n
    s = aligo_psd(f)[None]
    w = WH.inject_whiten(x, None, s, fs, 20.0, 1000.0)
    wk = np.fft.rfft(w, axis=-1)
    band = (f >= 20) & (f <= 1000)
    per_bin = np.mean(np.abs(wk[:, 0, band]) ** 2, axis=0) / n
    nb = band.sum()
    assert abs(per_bin.mean() - 1) < 4 / np.sqrt(reps * nb)
    assert np.abs(wk[:, 0, ~band]).max() < 1e-9
    frac = (2 * nb) / n                       # kept-band fraction of the N real degrees of freedom
    assert abs(w.var() / frac - 1) < 0.01 and abs(frac - 0.9572) < 5e-4


def test_unit_variance_with_welch_psd_is_biased_by_keff():
    # I-3: with a 63-segment Hann/50 % Welch estimate E[1/S_hat] = S^-1 K_eff/(K_eff-1) -> 1.017
    fs, n = 2048.0, 16384
    rng = np.random.Generator(np.random.Philox(31))
    vals = []
    for _ in range(6):
        bg = coloured_noise(rng, (1,), 131072, fs, dtype=np.float64)
        x = coloured_noise(rng, (4, 1), n, fs, dtype=np.float64)
        w = WH.inject_whiten(x, None, WE.welch(bg, fs, 4096), fs, 20.0, 1000.0)
        vals.append(w.var() / 0.9572)
    assert abs(np.mean(vals) - 1.0170) < 0.006


def test_gather_and_snr():
    strip = np.arange(40.0).reshape(2, 20)
    off = np.array([[0, 3], [12, 5]])
    g = WH.gather(strip, off, 8)
    assert np.all(g[1, 0] == np.arange(12, 20)) and np.all(g[0, 1] == 20 + np.arange(3, 11))
    # SNR scales as 1/distance and adds in quadrature over detectors
    k, n, fs = 129, 256, 256.0
    h = np.ones((1, 2, k), dtype=complex)
    s = np.ones((2, k))
    r1 = WH.optimal_snr(h, s, n, fs, 10.0, 100.0)
    assert abs(WH.optimal_snr(0.5 * h, s, n, fs, 10.0, 100.0) / r1 - 0.5) < 1e-15
    assert abs(r1 ** 2 - 2 * 4 * (fs / n) * 91) < 1e-9
