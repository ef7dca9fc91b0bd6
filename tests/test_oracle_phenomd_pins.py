"""Pins for the IMRPhenomD half of oracle.waveform that do not need lalsimulation.

The oracle types the aligned-spin post-Newtonian coefficients of ref. [32] in the
INDIVIDUAL-spin form (m1^2 chi1 + m2^2 chi2 and delta (m2 chi2 - m1 chi1) combinations, amplitude terms in chi1, chi2
and sqrt(1 - 4 eta)).  Appendix B of [32] prints the same coefficients in the (chi_s, chi_a, delta) form; the two
are different rational numbers multiplying different combinations, so a wrong digit or sign in either breaks the
identity.  Further pins: test-mass limits of the remnant fits, exchange symmetry of every coefficient at q != 1, and
bounds over a sweep of the Table-1 priors that a mistyped fit-table row violates.
"""
import numpy as np
import pytest

from oracle import fft as F
from oracle import waveform as W

PI = np.pi
CASES = [(0.3, 0.7, -0.4), (0.125, -0.9, 0.8), (0.6, 0.2, 0.95), (0.9, -0.5, 0.3), (0.45, 0.99, 0.99)]


def eta_of(q):
    return q / (1.0 + q) ** 2


def appendix_b_phase(eta, chi1, chi2, exchange=False):
    """[32] App. B: the spin-dependent TaylorF2 phasing coefficients phi_3 .. phi_7 in (chi_s, chi_a, delta),
    delta = sqrt(1 - 4 eta) (m1 >= m2).  Returns (phi3, phi4, phi5 [the factor of 1 + ln(pi M f)], spin part of phi6, phi7).
    exchange: the same binary with the bodies named the other way round (delta -> -delta, chi_a -> -chi_a)."""
    d = np.sqrt(1.0 - 4.0 * eta)
    xs, xa = 0.5 * (chi1 + chi2), 0.5 * (chi1 - chi2)
    if exchange:
        d, xa = -d, -xa
    phi3 = -16.0 * PI + 113.0 * d / 3.0 * xa + (113.0 / 3.0 - 76.0 * eta / 3.0) * xs
    phi4 = (15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta ** 2 / 72.0
            + (-405.0 / 8.0 + 200.0 * eta) * xa ** 2 - 405.0 / 4.0 * d * xa * xs + (-405.0 / 8.0 + 5.0 * eta / 2.0) * xs ** 2)
    phi5 = (38645.0 * PI / 756.0 - 65.0 * PI * eta / 9.0 + d * (-732985.0 / 2268.0 - 140.0 * eta / 9.0) * xa
            + (-732985.0 / 2268.0 + 24260.0 * eta / 81.0 + 340.0 * eta ** 2 / 9.0) * xs)
    phi6_spin = 2270.0 / 3.0 * PI * d * xa + (2270.0 * PI / 3.0 - 520.0 * PI * eta) * xs
    phi7 = (77096675.0 * PI / 254016.0 + 378515.0 * PI * eta / 1512.0 - 74045.0 * PI * eta ** 2 / 756.0
            + d * (-25150083775.0 / 3048192.0 + 26804935.0 * eta / 6048.0 - 1985.0 * eta ** 2 / 48.0) * xa
            + (-25150083775.0 / 3048192.0 + 10566655595.0 * eta / 762048.0 - 1042165.0 * eta ** 2 / 3024.0
               + 5345.0 * eta ** 3 / 36.0) * xs)
    return phi3, phi4, phi5, phi6_spin, phi7


def appendix_b_amp(eta, chi1, chi2, exchange=False):
    """[32] App. B: amplitude coefficients A_2 .. A_6 in (chi_s, chi_a, delta)."""
    d = np.sqrt(1.0 - 4.0 * eta)
    xs, xa = 0.5 * (chi1 + chi2), 0.5 * (chi1 - chi2)
    if exchange:
        d, xa = -d, -xa
    a2 = -323.0 / 224.0 + 451.0 * eta / 168.0
    a3 = (27.0 / 8.0 - 11.0 * eta / 6.0) * xs + 27.0 / 8.0 * d * xa
    a4 = (-27312085.0 / 8128512.0 - 1975055.0 * eta / 338688.0 + 105271.0 * eta ** 2 / 24192.0
          + (-81.0 / 32.0 + 8.0 * eta) * xa ** 2 - 81.0 / 16.0 * d * xa * xs + (-81.0 / 32.0 + 17.0 * eta / 8.0) * xs ** 2)
    a5 = (-85.0 * PI / 64.0 + 85.0 * PI * eta / 16.0 + d * xa * (285197.0 / 16128.0 - 1579.0 * eta / 4032.0)
          + xs * (285197.0 / 16128.0 - 15317.0 * eta / 672.0 - 2227.0 * eta ** 2 / 1008.0))
    a6 = (-177520268561.0 / 8583708672.0 + (545384828789.0 / 5007163392.0 - 205.0 * PI ** 2 / 48.0) * eta
          - 3248849057.0 * eta ** 2 / 178827264.0 + 34473079.0 * eta ** 3 / 6386688.0
          + xa ** 2 * (1614569.0 / 64512.0 - 1873643.0 * eta / 16128.0 + 2167.0 * eta ** 2 / 42.0)
          + xs ** 2 * (1614569.0 / 64512.0 - 61391.0 * eta / 1344.0 + 57451.0 * eta ** 2 / 4032.0)
          + (31.0 * PI / 12.0 - 7.0 * PI * eta / 3.0) * xs
          + d * xa * (31.0 * PI / 12.0 + xs * (1614569.0 / 32256.0 - 165961.0 * eta / 2688.0)))
    return a2, a3, a4, a5, a6


# ------------------------------- (a) spin terms of the phasing, q != 1, chi1 != chi2 ------------------------------

@pytest.mark.parametrize("q,chi1,chi2", CASES)
def test_pn_phase_spin_terms_equal_appendix_b_form(q, chi1, chi2):
    eta = eta_of(q)
    v, vl = W.pn_phase_coeffs(eta, chi1, chi2)
    v0, vl0 = W.pn_phase_coeffs(eta, 0.0, 0.0)
    phi3, phi4, phi5, phi6s, phi7 = appendix_b_phase(eta, chi1, chi2)
    assert abs(v[3] - phi3) < 1e-12 * abs(phi3)
    assert abs(v[4] - phi4) < 1e-12 * abs(phi4)
    # phi5 multiplies 1 + ln(pi M f) = 1 + 3 ln v: constant part and logarithmic part
    assert abs(v[5] - phi5) < 1e-12 * abs(phi5) and abs(vl[5] - 3.0 * phi5) < 1e-12 * abs(phi5)
    assert abs((v[6] - v0[6]) - phi6s) < 1e-11 * abs(phi6s) and vl[6] == vl0[6]
    assert abs(v[7] - phi7) < 1e-12 * abs(phi7)
    # nothing else carries spin
    assert v[0] == v0[0] and v[2] == v0[2] and np.all(vl[:5] == 0.0) and vl[7] == 0.0


def test_leading_spin_orbit_term_is_beta_of_ref33():
    """1.5PN: psi_3 = -16 pi + 4 beta with beta = sum_i (113/12 (m_i/M)^2 + 25/4 eta) chi_i (the spin-orbit parameter of
    [33]); 2PN: psi_4 = ... - 10 sigma with the black-hole quadrupole terms: third, per-body form of the same numbers."""
    for q, chi1, chi2 in CASES:
        eta = eta_of(q)
        m1, m2 = 1.0 / (1.0 + q), q / (1.0 + q)
        beta = (113.0 / 12.0 * m1 ** 2 + 25.0 / 4.0 * eta) * chi1 + (113.0 / 12.0 * m2 ** 2 + 25.0 / 4.0 * eta) * chi2
        v, _ = W.pn_phase_coeffs(eta, chi1, chi2)
        v0, _ = W.pn_phase_coeffs(eta, 0.0, 0.0)
        assert abs(v[3] - (-16.0 * PI + 4.0 * beta)) < 1e-12
        sigma = 79.0 / 8.0 * eta * chi1 * chi2 + 81.0 / 16.0 * (m1 ** 2 * chi1 ** 2 + m2 ** 2 * chi2 ** 2)
        assert abs((v[4] - v0[4]) + 10.0 * sigma) < 1e-12


# ------------------------------- (c) amplitude coefficients ------------------------------------------------------

@pytest.mark.parametrize("q,chi1,chi2", CASES)
def test_amp_pn_coeffs_equal_appendix_b_form(q, chi1, chi2):
    eta = eta_of(q)
    got = W.amp_pn_coeffs(eta, chi1, chi2)
    ref = appendix_b_amp(eta, chi1, chi2)
    assert got[0] == pytest.approx((-969.0 + 1804.0 * eta) / 672.0, rel=1e-15)
    for g, r in zip(got, ref):
        assert abs(g - r) < 1e-12 * max(1.0, abs(r))


def test_amp_and_phase_coeffs_invariant_under_exchange_of_the_bodies():
    """(m1, chi1) <-> (m2, chi2) is delta -> -delta, chi_a -> -chi_a: the test's own copy of the exchanged (chi_s, chi_a,
    delta) expressions equals the oracle's coefficients at q != 1 (the oracle derives sqrt(1 - 4 eta) itself, so the
    exchange is applied on the test's side); at q = 1 swapping the spins changes nothing."""
    for q, chi1, chi2 in CASES:
        eta = eta_of(q)
        for g, r in zip(W.amp_pn_coeffs(eta, chi1, chi2), appendix_b_amp(eta, chi1, chi2, exchange=True)):
            assert abs(g - r) < 1e-12 * max(1.0, abs(r))
        v, vl = W.pn_phase_coeffs(eta, chi1, chi2)
        v0, _ = W.pn_phase_coeffs(eta, 0.0, 0.0)
        phi3, phi4, phi5, phi6s, phi7 = appendix_b_phase(eta, chi1, chi2, exchange=True)
        got = [v[3], v[4], v[5], v[6] - v0[6], v[7]]
        for g, r in zip(got, [phi3, phi4, phi5, phi6s, phi7]):
            assert abs(g - r) < 1e-11 * max(1.0, abs(r))
    for chi1, chi2 in [(0.6, -0.4), (-0.9, 0.3)]:
        assert np.allclose(W.amp_pn_coeffs(0.25, chi1, chi2), W.amp_pn_coeffs(0.25, chi2, chi1), rtol=1e-13, atol=1e-13)
        pa, la = W.pn_phase_coeffs(0.25, chi1, chi2)
        pb, lb = W.pn_phase_coeffs(0.25, chi2, chi1)
        assert np.allclose(pa, pb, rtol=1e-13) and np.allclose(la, lb, rtol=1e-13)


# ------------------------------- (b) remnant fits: limits the mathematics fixes ------------------------------------

def kerr_isco_energy(a):
    """Specific energy of the prograde equatorial ISCO of a Kerr hole of spin a (Bardeen, Press & Teukolsky 1972)."""
    z1 = 1.0 + np.cbrt(1.0 - a * a) * (np.cbrt(1.0 + a) + np.cbrt(1.0 - a))
    z2 = np.sqrt(3.0 * a * a + z1 * z1)
    r = 3.0 + z2 - np.sign(a) * np.sqrt((3.0 - z1) * (3.0 + z1 + 2.0 * z2))
    return np.sqrt(1.0 - 2.0 / (3.0 * r))


def test_final_spin_and_radiated_energy_test_mass_limits():
    for chi1 in (-0.9, -0.3, 0.0, 0.5, 0.95):
        for chi2 in (-0.8, 0.0, 0.7):
            # a test body changes nothing: the remnant keeps the spin of the heavy hole, nothing is radiated
            assert abs(W.final_spin(1e-9, chi1, chi2) - chi1) < 1e-7
            assert abs(W.e_rad(1e-9, chi1, chi2)) < 1e-9
    # first order in eta: E_rad / eta -> 1 - E_ISCO(chi1), Schwarzschild 1 - sqrt(8/9) = 0.0572 (the fit is a few per cent off)
    assert abs(W.e_rad(1e-6, 0.0, 0.0) / 1e-6 / (1.0 - np.sqrt(8.0 / 9.0)) - 1.0) < 0.03
    for a in (-0.9, -0.5, 0.5, 0.8):
        assert abs(W.e_rad(1e-6, a, 0.0) / 1e-6 / (1.0 - kerr_isco_energy(a)) - 1.0) < 0.15
    # ... and d a_f / d eta -> orbital angular momentum of the ISCO minus 2 chi (first-order spin change of the hole);
    # at chi = 0 that is L_ISCO = sqrt(12) = 3.4641
    assert abs((W.final_spin(1e-6, 0.0, 0.0) - 0.0) / 1e-6 - np.sqrt(12.0)) < 1e-3


def test_remnant_monotone_in_spin_and_bounded():
    chis = np.linspace(-0.99, 0.99, 41)
    for q in (1.0, 0.5, 0.125):
        eta = eta_of(q)
        af = np.array([W.final_spin(eta, c, c) for c in chis])
        er = np.array([W.e_rad(eta, c, c) for c in chis])
        assert np.all(np.diff(af) > 0) and np.all(np.diff(er) > 0)        # more aligned spin: later plunge (Kerr ISCO)
        assert np.all(np.abs(af) < 1.0) and np.all((er > 0) & (er < 0.12))
        frd = np.array([W.ringdown_freqs(eta, c, c)[0] for c in chis])
        fdm = np.array([W.ringdown_freqs(eta, c, c)[1] for c in chis])
        assert np.all(np.diff(frd) > 0)                                    # the Kerr (2,2,0) frequency rises with spin
        assert np.all((fdm > 0.004) & (fdm < 0.02)) and np.all(frd / fdm > 3.0)      # quality factor Q = f_RD / (2 f_damp) > 1.5
    # mass-ratio trend at zero spin: a_f and E_rad grow with eta up to the equal-mass values 0.686 / 4.8 %
    etas = np.linspace(0.02, 0.25, 24)
    assert np.all(np.diff([W.final_spin(e, 0, 0) for e in etas]) > 0)
    assert np.all(np.diff([W.e_rad(e, 0, 0) for e in etas]) > 0)


# ------------------------------- (d) bounds over the Table-1 priors that a mistyped table row violates -------------

def prior_sweep(count, seed):
    rng = np.random.Generator(np.random.Philox(seed))
    q = rng.uniform(0.125, 1.0, count)
    return q, rng.uniform(-0.99, 0.99, count), rng.uniform(-0.99, 0.99, count)


def test_fit_terms_stay_corrections_over_the_prior():
    """The fitted terms (sigma, rho, v2, gamma, beta, alpha rows of the table of [32]) are corrections to known physics; a
    wrong digit or a swapped row makes them dominate.  Bounds are ~2x what the table as transcribed gives over 1000 draws."""
    q, c1, c2 = prior_sweep(1000, 123)
    f_ins = np.linspace(0.0035, 0.018, 200)
    basis = np.vstack([np.ones_like(f_ins), f_ins]).T
    g = np.linspace(0.002, 0.2, 2000)
    for i in range(len(q)):
        eta = eta_of(q[i])
        pd = W.PhenomD(eta, c1[i], c2[i])
        pd0 = W.PhenomD(eta, c1[i], c2[i], sigma_scale=0.0)
        # sigma terms: beyond a time and phase shift (a + b f) they change the inspiral phase by a few radians
        diff = pd.phi_ins(f_ins) - pd0.phi_ins(f_ins)
        co = np.linalg.lstsq(basis, diff, rcond=None)[0]
        assert np.abs(diff - basis @ co).max() < 10.0
        # rho terms: the inspiral amplitude at its upper end stays within 30 % of the PN series
        a2, a3, a4, a5, a6 = pd.amp_a
        x = np.cbrt(np.pi * 0.014)
        pn = 1.0 + a2 * x ** 2 + a3 * x ** 3 + a4 * x ** 4 + a5 * x ** 5 + a6 * x ** 6
        assert 0.7 < pd.amp_ins(0.014) / pn < 1.05
        # the full amplitude: positive, its bracket (A f^(7/6)) has ONE maximum, f^2 |h| peaks just below the ringdown
        amp = pd.amplitude(g)
        assert np.all(amp > 0.0) and np.all(np.isfinite(amp))
        br = amp * g ** (7.0 / 6.0)
        d = np.diff(br)
        assert np.sum((d[:-1] > 0) & (d[1:] <= 0)) == 1
        assert 0.5 < g[np.argmax(br * g)] / pd.f_rd < 1.1
        assert 0.8 < pd.f_peak / pd.f_rd < 1.0
        # alpha / beta rows: the group delay (d phi / df - t0) / 2 pi around the ringdown stays within tens of M of the peak
        assert np.all(np.isfinite(pd.phase(g)))
        fm = np.linspace(0.5 * pd.f_rd, 1.2 * pd.f_rd, 100)
        tau = (pd.dphi_mr_raw(fm) + pd.c2_mr - pd.t0) / (2.0 * np.pi)
        assert -80.0 < tau.min() and tau.max() < 40.0


def test_time_domain_peak_sits_at_tc_over_the_prior():
    """t_c is the time of the amplitude peak (reading R-W1: t0 = d phi_MR / df at f_peak): over 40 draws of the priors the
    envelope of the band-limited time series peaks 5 .. 25 M before t_c (never after, never further)."""
    from oracle.constants import MTSUN_SI
    rng = np.random.Generator(np.random.Philox(321))
    n, fs = 16384, 2048.0
    for _ in range(40):
        mc, q = rng.uniform(10.0, 100.0), rng.uniform(0.125, 1.0)
        c1, c2 = rng.uniform(-0.99, 0.99, 2)
        tc = rng.uniform(5.5, 6.5)
        row = np.array([mc, q, c1, c2, 1000.0, 0.3, 0.2, tc, 1.0, 0.5, 0.7])
        h0 = W.imrphenomd_h0(row, n // 2 + 1, n / fs, 20.0, 1000.0)
        spec = np.zeros(n, dtype=np.complex128)
        spec[:n // 2 + 1] = h0 * fs
        env = np.abs(np.fft.ifft(spec))                       # analytic signal (positive frequencies only)
        ms = W.masses(mc, q)[0] * MTSUN_SI
        dt = np.argmax(env) / fs - tc
        assert -30.0 * ms - 1.0 / fs < dt < 2.0 * ms + 1.0 / fs
