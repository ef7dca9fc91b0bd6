"""Property-based checks of the oracle on tiny inputs (hypothesis): invariants that hold for ANY input, so that a
dropped term, a wrong sign or a transposed index somewhere in the oracle shows up on some drawn example.
SURVEY.md section 4 tier (3); BASELINE.json north_star invariants (Parseval, psi-independence, light-travel bound,
linearity of injection)."""
import numpy as np
from hypothesis import given, settings, strategies as st

from oracle import fft as F
from oracle import project as OP
from oracle import waveform as OW
from oracle import welch as WE
from oracle import whiten as WH
from oracle.constants import C_SI, DETECTORS

CFG = dict(max_examples=30, deadline=None)
angles = st.floats(min_value=-10.0, max_value=10.0, allow_nan=False)


@settings(**CFG)
@given(st.integers(min_value=2, max_value=9), st.integers(min_value=0, max_value=2 ** 31 - 1))
def test_fft_equals_numpy_and_parseval(log2n, seed):
    n = 1 << log2n
    x = np.random.default_rng(seed).standard_normal(n)
    xk = F.rfft(x)
    assert np.abs(xk - np.fft.rfft(x)).max() <= 1e-11 * max(1.0, np.abs(xk).max())
    assert np.abs(F.dft_naive(x.astype(complex))[: n // 2 + 1] - xk).max() <= 1e-10 * max(1.0, np.abs(xk).max())
    energy = (np.abs(xk[0]) ** 2 + 2 * np.sum(np.abs(xk[1:-1]) ** 2) + np.abs(xk[-1]) ** 2) / n
    assert abs(energy - np.sum(x * x)) <= 1e-10 * max(1.0, np.sum(x * x))
    assert np.abs(F.irfft(xk, n) - x).max() <= 1e-12 * max(1.0, np.abs(x).max())


@settings(**CFG)
@given(angles, angles, angles, angles, angles, st.integers(min_value=0, max_value=2))
def test_antenna_pattern_invariants(ra, dec, psi, psi2, gmst, det):
    dd = DETECTORS[det]
    fp, fc, dt = OP.response(ra, dec, psi, gmst, dd["r"], dd["x"], dd["y"])
    fp2, fc2, dt2 = OP.response(ra, dec, psi2, gmst, dd["r"], dd["x"], dd["y"])
    assert abs((fp * fp + fc * fc) - (fp2 * fp2 + fc2 * fc2)) < 1e-12          # independent of the polarisation angle
    assert fp * fp + fc * fc <= 1.0 + 1e-9
    assert dt == dt2 and abs(dt) <= np.linalg.norm(dd["r"]) / C_SI + 1e-15      # delay bounded by the light-travel time
    fp3, fc3, _ = OP.response(ra, dec, psi + np.pi / 2, gmst, dd["r"], dd["x"], dd["y"])
    assert abs(fp3 + fp) < 1e-12 and abs(fc3 + fc) < 1e-12                      # psi -> psi + pi/2 flips both
    fp4, fc4, dt4 = OP.response(ra + 0.37, dec, psi, gmst + 0.37, dd["r"], dd["x"], dd["y"])
    assert abs(fp4 - fp) < 1e-12 and abs(fc4 - fc) < 1e-12 and abs(dt4 - dt) < 1e-15   # only gmst - ra matters
    for other in range(3):
        _, _, dto = OP.response(ra, dec, psi, gmst, DETECTORS[other]["r"], DETECTORS[other]["x"], DETECTORS[other]["y"])
        assert abs(dt - dto) <= np.linalg.norm(dd["r"] - DETECTORS[other]["r"]) / C_SI + 1e-15


@settings(**CFG)
@given(st.integers(min_value=0, max_value=2 ** 31 - 1), st.floats(min_value=-3, max_value=3), st.floats(min_value=-3, max_value=3),
       st.sampled_from([64, 128, 256]))
def test_whitening_is_linear_and_band_limited(seed, a, b, n):
    rng = np.random.default_rng(seed)
    fs = 64.0
    k = n // 2 + 1
    psd = (0.5 + rng.random((1, k)))
    x1, x2 = rng.standard_normal((1, 1, n)), rng.standard_normal((1, 1, n))
    h = (rng.standard_normal((1, 1, k)) + 1j * rng.standard_normal((1, 1, k)))
    f_lo, f_hi = 4.0, 20.0
    w = lambda x, hh: WH.inject_whiten(x, hh, psd, fs, f_lo, f_hi)
    lhs = w(a * x1 + b * x2, (a + b) * h)
    rhs = a * w(x1, h) + b * w(x2, h)
    assert np.abs(lhs - rhs).max() <= 1e-10 * max(1.0, np.abs(rhs).max())
    yk = np.fft.rfft(lhs[0, 0])
    f = np.arange(k) * fs / n
    assert np.abs(yk[(f < f_lo) | (f > f_hi)]).max() <= 1e-9 * max(1.0, np.abs(yk).max())
    # the frequency-domain injection is the time-domain addition of the circular inverse transform (R-I1)
    s_t = fs * F.irfft(h[0, 0], n)
    assert np.abs(w(x1 + s_t, None) - w(x1, h)).max() <= 1e-9 * max(1.0, np.abs(lhs).max())


@settings(**CFG)
@given(st.integers(min_value=0, max_value=2 ** 31 - 1), st.floats(min_value=0.1, max_value=50.0), st.sampled_from([32, 64]),
       st.integers(min_value=0, max_value=5), st.sampled_from(["mean", "median"]))
def test_welch_scaling_and_segment_count(seed, scale, nperseg, extra, average):
    rng = np.random.default_rng(seed)
    n_bg = nperseg * 4 + extra * 7
    x = rng.standard_normal(n_bg)
    p1 = WE.welch(x, 64.0, nperseg, average=average)
    p2 = WE.welch(scale * x + 5.0, 64.0, nperseg, average=average)            # detrended: the offset is removed
    assert np.abs(p2[1:] - scale * scale * p1[1:]).max() <= 1e-9 * max(1e-30, np.abs(p2).max())
    assert np.all(p1 >= 0)
    # samples beyond the last full segment do not enter (R-S1)
    nseg = (n_bg - nperseg) // (nperseg // 2) + 1
    used = (nseg - 1) * (nperseg // 2) + nperseg
    x2 = x.copy()
    x2[used:] += 100.0
    assert np.array_equal(WE.welch(x2, 64.0, nperseg, average=average), p1)


@settings(**CFG)
@given(st.floats(min_value=10.0, max_value=100.0), st.floats(min_value=0.125, max_value=1.0), st.floats(min_value=-0.99, max_value=0.99),
       st.floats(min_value=-0.99, max_value=0.99), st.floats(min_value=100.0, max_value=3000.0), angles, angles,
       st.sampled_from([OW.TAYLORF2, OW.IMRPHENOMD]))
def test_waveform_symmetries(mc, q, c1, c2, dist, theta, phi, approx):
    n, fs = 1024, 2048.0
    p = np.array([[mc, q, c1, c2, dist, theta, phi, 0.3, 0.0, 0.0, 0.0]])
    hp, hc, fl = OW.waveform_fd(approx, p, n, fs, 20.0, 1000.0)
    assert fl[0] == 0 and np.all(np.isfinite(hp)) and np.all(np.isfinite(hc))
    assert hp[0, 0] == 0 and hp[0, -1] == 0                                     # DC and Nyquist always zero (R-W7)
    p2 = p.copy(); p2[0, 6] += np.pi                                            # phi_c -> phi_c + pi: unchanged (R-W5)
    hp2, _, _ = OW.waveform_fd(approx, p2, n, fs, 20.0, 1000.0)
    assert np.abs(hp2 - hp).max() <= 1e-9 * max(np.abs(hp).max(), 1e-300)
    p3 = p.copy(); p3[0, 4] *= 2.0                                              # twice the distance: half the strain
    hp3, _, _ = OW.waveform_fd(approx, p3, n, fs, 20.0, 1000.0)
    assert np.abs(2.0 * hp3 - hp).max() <= 1e-12 * max(np.abs(hp).max(), 1e-300)
    ci = np.cos(theta)                                                          # hx = -i cos(i) h0, h+ = (1 + cos^2 i)/2 h0 (R-W6)
    assert np.abs(hc * 0.5 * (1 + ci * ci) - (-1j) * ci * hp).max() <= 1e-12 * max(np.abs(hp).max(), 1e-300)
