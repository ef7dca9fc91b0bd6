"""Pins for the oracle functions of the SURVEY.md 8(f) rows: time-domain waveform output, the two data views
(PAPER.md:93, :117), median-averaged Welch and the time-truncated whitening filter.  Each pin is something
other than the oracle's own formula: a library routine of a different kind (scipy.signal.hilbert,
scipy.signal.welch(average='median'), numpy.convolve), a closed form, a symmetry or a Monte-Carlo estimate."""
import numpy as np
import pytest
import scipy.signal

from oracle import fft as F
from oracle import project as OP
from oracle import views as OV
from oracle import waveform as OW
from oracle import welch as WE
from oracle import whiten as WH
from oracle.constants import MTSUN_SI
from workloads import aligo_psd, coloured_noise, draw_params

FS, N = 2048.0, 8192


def _params(t_c=2.5, mc=20.0, q=0.8, theta=0.7):
    return np.array([[mc, q, 0.0, 0.0, 400.0, theta, 0.3, t_c, 1.0, -0.4, 0.9]])


# ---------------------------------------------------------------- time-domain waveform
@pytest.mark.parametrize("approx", [OW.TAYLORF2, OW.IMRPHENOMD])
def test_td_parseval(approx):
    p = _params()
    hp_t, hc_t, _ = OW.waveform_td(approx, p, N, FS, 20.0, 1000.0)
    hp, hc, _ = OW.waveform_fd(approx, p, N, FS, 20.0, 1000.0)
    df = FS / N
    for ht, hf in ((hp_t, hp), (hc_t, hc)):
        lhs = np.sum(ht ** 2) / FS                               # integral of h(t)^2 dt
        rhs = 2.0 * np.sum(np.abs(hf[:, 1:-1]) ** 2) * df         # 2 * integral over f > 0 of |h~|^2 df
        assert abs(lhs / rhs - 1) < 1e-12


def test_td_face_on_cross_is_hilbert_transform_of_plus():
    # iota = 0: hx~ = -i h+~ for f > 0, i.e. hx(t) is the Hilbert transform of h+(t)
    p = _params(theta=0.0)
    hp_t, hc_t, _ = OW.waveform_td(OW.IMRPHENOMD, p, N, FS, 20.0, 1000.0)
    ana = scipy.signal.hilbert(hp_t[0])
    assert np.abs(ana.imag - hc_t[0]).max() < 1e-9 * np.abs(hp_t).max()
    assert np.abs(ana.real - hp_t[0]).max() < 1e-12 * np.abs(hp_t).max()


def test_td_whole_sample_shift_is_a_roll():
    a, _, _ = OW.waveform_td(OW.IMRPHENOMD, _params(t_c=2.5), N, FS, 20.0, 1000.0)
    b, _, _ = OW.waveform_td(OW.IMRPHENOMD, _params(t_c=2.5 + 37 / FS), N, FS, 20.0, 1000.0)
    assert np.abs(np.roll(a[0], 37) - b[0]).max() < 1e-9 * np.abs(a).max()


def test_td_instantaneous_frequency_follows_newtonian_chirp():
    # low-mass TaylorF2: zero crossings of h+(t) a time tau before t_c are spaced by 1/(2 f(tau)),
    # f(tau) = (5 / (256 tau))^(3/8) (G Mc / c^3)^(-5/8) / pi  (textbook Newtonian chirp)
    mc, t_c, n = 12.0, 7.0, 16384
    p = np.array([[mc, 1.0, 0, 0, 400.0, 0.0, 0.0, t_c, 0, 0, 0]])
    h, _, _ = OW.waveform_td(OW.TAYLORF2, p, n, FS, 20.0, 1000.0)
    t = np.arange(n) / FS
    for tau in (2.0, 1.0, 0.5):
        sel = (t > t_c - tau - 0.1) & (t < t_c - tau + 0.1)
        x = h[0, sel]
        crossings = np.sum(np.signbit(x[1:]) != np.signbit(x[:-1]))
        f_meas = crossings / 2.0 / 0.2
        f_newt = (5.0 / (256.0 * tau)) ** 0.375 * (mc * MTSUN_SI) ** -0.625 / np.pi
        assert abs(f_meas / f_newt - 1) < 0.08, (tau, f_meas, f_newt)   # PN corrections are a few per cent here


# ---------------------------------------------------------------- two views
def _view_inputs(batch=3, n=4096):
    rng = np.random.Generator(np.random.Philox(77))
    par = draw_params(rng, batch, t_c=(1.0, 1.2))
    noise = coloured_noise(rng, (batch, 2), n, FS, dtype=np.float64)
    psd = np.stack([aligo_psd(np.arange(n // 2 + 1) * FS / n)] * 2)
    return par, noise, psd


def test_views_zero_shift_identical_and_noise_cancels():
    par, noise, psd = _view_inputs()
    n = noise.shape[-1]
    d, d2 = OV.two_views(OW.IMRPHENOMD, par, np.zeros(3), noise, psd, 0.0, [0, 1], FS, 20.0, 1000.0)
    assert np.array_equal(d, d2)
    shift = np.array([0.31, 0.9, 0.004])
    d, d2 = OV.two_views(OW.IMRPHENOMD, par, shift, noise, psd, 0.0, [0, 1], FS, 20.0, 1000.0)
    e, e2 = OV.two_views(OW.IMRPHENOMD, par, shift, 0.0 * noise, psd, 0.0, [0, 1], FS, 20.0, 1000.0)
    # same background in both views: the difference of the views contains no noise
    assert np.abs((d - d2) - (e - e2)).max() < 1e-9 * np.abs(d).max()
    assert np.abs(d - d2).max() > 1e-3                      # and the views do differ


def test_views_whole_sample_shift_rolls_the_signal_part():
    par, noise, psd = _view_inputs()
    shift = np.array([100, 2048, 1]) / FS
    d, d2 = OV.two_views(OW.IMRPHENOMD, par, shift, noise, psd, 0.0, [0, 1], FS, 20.0, 1000.0)
    bg = WH.inject_whiten(noise, None, psd, FS, 20.0, 1000.0)
    for b, m in enumerate((100, 2048, 1)):
        s1, s2 = d[b] - bg[b], d2[b] - bg[b]
        assert np.abs(np.roll(s1, m, axis=-1) - s2).max() < 1e-8 * max(np.abs(s1).max(), 1e-30)


# ---------------------------------------------------------------- median Welch
def test_median_bias_closed_forms():
    for n in (1, 3, 9, 63):
        alt = sum((-1.0) ** (i + 1) / i for i in range(1, n + 1))
        assert abs(WE.median_bias(n) - alt) < 1e-14
    assert WE.median_bias(1) == 1.0
    assert abs(WE.median_bias(2) - 1.0) < 1e-15             # mean of two = their midpoint
    assert abs(WE.median_bias(100001) - np.log(2.0)) < 1e-5


@pytest.mark.parametrize("nseg", [4, 10, 64])
def test_median_bias_even_monte_carlo(nseg):
    x = np.random.default_rng(nseg).exponential(size=(200000, nseg))
    est = np.median(x, axis=1).mean()
    assert abs(est / WE.median_bias(nseg) - 1) < 4e-3


@pytest.mark.parametrize("detrend", [0, 1])
@pytest.mark.parametrize("n_bg,nperseg", [(4096 + 256, 512), (131072, 4096)])      # 15 and 63 segments (odd)
def test_welch_median_matches_scipy_for_odd_segment_counts(n_bg, nperseg, detrend):
    x = np.random.default_rng(n_bg).standard_normal((2, n_bg)) * 3.0 + 0.7
    got = WE.welch(x, 2048.0, nperseg, detrend=detrend, average="median")
    _, ref = scipy.signal.welch(x, 2048.0, "hann", nperseg, nperseg // 2, detrend="constant" if detrend else False,
                                scaling="density", average="median")
    assert np.abs(got - ref).max() <= 1e-12 * ref.max()


def test_welch_median_level_and_glitch_robustness():
    fs, s = 2048.0, 3.0
    x = np.random.default_rng(5).standard_normal(1 << 18) * s
    for nperseg in (1024, 2048):                             # 511 (odd) and 255 (odd) segments
        med = WE.welch(x, fs, nperseg, detrend=0, average="median")
        assert abs(med[5:-5].mean() / (2 * s * s / fs) - 1) < 0.01
    med_even = WE.welch(x[: 1024 * 32 + 512], fs, 1024, detrend=0, average="median")   # 64 segments (even)
    assert abs(med_even[5:-5].mean() / (2 * s * s / fs) - 1) < 0.03
    y = x.copy()
    y[100000:100040] += 400.0                                # a loud transient
    mean_g = WE.welch(y, fs, 1024, detrend=0)
    med_g = WE.welch(y, fs, 1024, detrend=0, average="median")
    level = 2 * s * s / fs
    assert mean_g[5:200].mean() / level > 1.5                # the mean is pulled up
    assert abs(med_g[5:200].mean() / level - 1) < 0.03       # the median is not


# ---------------------------------------------------------------- truncated whitening filter
def test_fir_filter_is_real_even_and_has_finite_support():
    n, fdur = 4096, 0.5
    psd = aligo_psd(np.arange(n // 2 + 1) * FS / n)[None]
    wf = WH.fir_truncated_filter(psd, n, FS, 20.0, 1000.0, fdur)
    q = F.irfft(wf[0].astype(complex), n)
    m = np.minimum(np.arange(n), n - np.arange(n))
    ntaps = int(fdur * FS)
    assert np.abs(q[m >= ntaps // 2]).max() < 1e-12 * np.abs(q).max()
    assert np.abs(q[1:] - q[1:][::-1]).max() < 1e-12 * np.abs(q).max()
    # lag 0 is untouched by the taper and carries the mean of the untruncated response
    w0 = WH.whitening_filter(psd, n, FS, 20.0, 1000.0)[0]
    assert abs(q[0] / F.irfft(w0.astype(complex), n)[0] - 1) < 1e-12


def test_fir_whitening_equals_linear_convolution_inside_the_crop():
    rng = np.random.default_rng(3)
    n, fdur = 2048, 0.25
    ntaps = int(fdur * FS)
    pad = ntaps // 2
    x = rng.standard_normal((2, 1, n))
    psd = (aligo_psd(np.arange(n // 2 + 1) * FS / n) * (1 + 0.3 * rng.random(n // 2 + 1)))[None]
    got = WH.inject_whiten_fir(x, None, psd, FS, 20.0, 1000.0, fdur)
    assert got.shape == (2, 1, n - ntaps)
    wf = WH.fir_truncated_filter(psd, n, FS, 20.0, 1000.0, fdur)[0]
    q = np.fft.irfft(wf, n)
    taps = np.concatenate([q[n - pad + 1:], q[:pad]])        # lags -(pad-1) .. +(pad-1)
    for b in range(2):
        lin = np.convolve(x[b, 0], taps, mode="full")        # lin[i] = sum_m taps[m] x[i - m]
        ref = lin[pad - 1 + pad: pad - 1 + n - pad]          # output sample j <-> lin[j + pad - 1]
        assert np.abs(got[b, 0] - ref).max() < 1e-9 * np.abs(ref).max()
    # hence the cropped output does not depend on the samples a circular filter would wrap around:
    x2 = x.copy()
    x2[..., :1] += 50.0
    x2[..., -1:] -= 70.0
    got2 = WH.inject_whiten_fir(x2, None, psd, FS, 20.0, 1000.0, fdur)
    assert np.abs(got2 - got).max() < 1e-9 * np.abs(got).max()


def test_fir_whitened_noise_variance_and_signal_linearity():
    rng = np.random.Generator(np.random.Philox(9))
    n = 16384
    x = coloured_noise(rng, (64, 1), n, FS, dtype=np.float64)
    psd = aligo_psd(np.arange(n // 2 + 1) * FS / n)[None]
    y = WH.inject_whiten_fir(x, None, psd, FS, 20.0, 1000.0, 1.0)
    kept = (1000.0 - 20.0) / (FS / 2)
    assert abs(y.var() / kept - 1) < 0.02                    # smooth PSD: truncation changes little
    par = draw_params(rng, 1, t_c=(5.0, 5.1))
    hp, hc, _ = OW.waveform_fd(OW.IMRPHENOMD, par, n, FS, 20.0, 1000.0)
    h_det, _ = OP.project(hp, hc, par, 0.0, [0], n, FS)
    a = WH.inject_whiten_fir(x[:1], h_det, psd, FS, 20.0, 1000.0, 1.0)
    s = WH.inject_whiten_fir(0 * x[:1], h_det, psd, FS, 20.0, 1000.0, 1.0)
    assert np.abs(a - (y[:1] + s)).max() < 1e-9 * np.abs(a).max()


# ---------------------------------------------------------------- sine-Gaussian burst
def _sg(f0=250.0, q=9.0, amp=1e-21, iota=0.6, phi=0.4, t0=2.0):
    return np.array([f0, q, 0.0, 0.0, amp, iota, phi, t0, 1.0, -0.4, 0.9])


@pytest.mark.parametrize("f0,q", [(250.0, 9.0), (80.0, 5.0), (600.0, 30.0)])
def test_sine_gaussian_fd_model_is_the_fourier_transform_of_the_td_definition(f0, q):
    # independent route: sample the time-domain closed form and take numpy's FFT; X[k]/fs approximates the continuous
    # Fourier transform (the Gaussian is far from the segment edges and far below Nyquist)
    p = _sg(f0=f0, q=q)
    t = np.arange(N) / FS
    hp_t, hc_t = OW.sine_gaussian_td(p, t)
    hp, hc, flags = OW.waveform_fd(OW.SINE_GAUSSIAN, p[None], N, FS, 1.0, 1023.0)
    assert flags[0] == 0
    for ht, hf in ((hp_t, hp[0]), (hc_t, hc[0])):
        ref = np.fft.rfft(ht) / FS
        scale = np.abs(ref).max()
        # the dropped mirror term is at most e^(-Q^2/2) of the peak (reached as f -> 0)
        assert np.abs(hf[5:-5] - ref[5:-5]).max() < max(3.0 * np.exp(-0.5 * q * q), 1e-9) * scale
    # duration and central frequency are what the parameters say ("central frequency or duration")
    tau = q / (np.sqrt(2.0) * np.pi * f0)
    env2 = hp_t ** 2 + (hc_t * (0.5 * (1 + np.cos(0.6) ** 2)) / np.cos(0.6)) ** 2
    t_mean = np.sum(t * env2) / np.sum(env2)
    assert abs(t_mean - 2.0) < 1e-6
    assert abs(np.sqrt(np.sum((t - t_mean) ** 2 * env2) / np.sum(env2)) / (tau / 2.0) - 1) < 1e-6
    kpk = np.argmax(np.abs(hp[0]))
    assert abs(kpk * FS / N - f0) <= FS / N


def test_sine_gaussian_band_flags_and_td_output():
    p = np.stack([_sg(), _sg(q=-1.0), _sg(amp=0.0), _sg(f0=np.nan)])
    hp, hc, flags = OW.waveform_fd(OW.SINE_GAUSSIAN, p, N, FS, 200.0, 300.0)
    assert list(flags) == [0, 1, 1, 1]
    assert np.all(hp[1:] == 0) and np.all(hc[1:] == 0)
    f = np.arange(N // 2 + 1) * FS / N
    assert np.all(hp[0][(f < 200.0) | (f > 300.0)] == 0) and hp[0][f == 200.0] != 0 and hp[0][f == 300.0] != 0
    # the time-domain output call reproduces the closed form (full band)
    hp_t, hc_t, _ = OW.waveform_td(OW.SINE_GAUSSIAN, _sg()[None], N, FS, 1.0, 1023.0)
    a, b = OW.sine_gaussian_td(_sg(), np.arange(N) / FS)
    assert np.abs(hp_t[0] - a).max() < 1e-9 * np.abs(a).max()
    assert np.abs(hc_t[0] - b).max() < 1e-9 * np.abs(a).max()
