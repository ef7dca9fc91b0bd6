"""Pins for oracle.waveform (W-1..W-11; BASELINE north_star check
"TaylorF2 closed-form phase at fixed frequencies")."""
import numpy as np
import pytest

from oracle import constants as C
from oracle import fft as F
from oracle import phenomd_coeffs as T
from oracle import waveform as W
from workloads import aligo_psd

from conftest import read_golden

G = read_golden("taylorf2_worked_examples.txt")


def P(mc=26.0, q=1.0, c1=0.0, c2=0.0, d=1000.0, th=0.3, phic=0.0, tc=0.0, ra=1.0, dec=0.5, psi=0.7):
    return np.array([mc, q, c1, c2, d, th, phic, tc, ra, dec, psi], dtype=np.float64)


# ------------------------------- TaylorF2 -------------------------------------------------

@pytest.mark.parametrize("tag,mc,q,dist", [("fig1", 26.0, 1.0, 1000.0), ("b", 10.0, 0.25, 200.0)])
def test_taylorf2_worked_examples(tag, mc, q, dist):
    mtot = W.masses(mc, q)[0]
    assert abs(mtot - G[tag + "_mtot"][0]) < 1e-9
    assert abs(W.f_isco(mtot) - G[tag + "_fisco"][0]) < 1e-6
    assert abs(W.taylorf2_amp0(mc, dist) / G[tag + "_a0"][0] - 1) < 1e-11
    assert abs(W.chirp_time(20.0, mc) - G[tag + "_tau20"][0]) < 1e-6
    f = np.array(G[tag + "_freqs"])
    psi = W.taylorf2_phase(f, mc, q)
    assert np.abs(psi - np.array(G[tag + "_psi"])).max() < 2e-9
    if tag == "fig1":
        amp = W.taylorf2_amp0(mc, dist) * f ** (-7.0 / 6.0)
        assert np.abs(amp / np.array(G["fig1_amp"]) - 1).max() < 1e-9


def test_taylorf2_leading_order_is_newtonian_chirp():
    # t(f) = (1/2pi) dPsi/df -> t_c - tau(f) as v -> 0: check the 0PN term through its f^(-8/3) scaling
    mc, q = 1e-3, 1.0          # tiny mass -> v tiny at these f -> PN corrections negligible
    f = np.array([20.0, 40.0])
    e = 1e-4
    dpsi = (W.taylorf2_phase(f + e, mc, q) - W.taylorf2_phase(f - e, mc, q)) / (2 * e)
    tau = W.chirp_time(f, mc)
    assert np.abs(-dpsi / (2 * np.pi) / tau - 1).max() < 2e-3


def test_group_delay_monotone_and_approaches_tc():
    # stationary phase: t(f) = (1/2pi) dPsi/df = -(1/2pi) d arg(h0)/df rises monotonically towards t_c
    # (t_c = 0 here so that the per-bin phase step stays below pi and unwrap is safe)
    h0 = W.taylorf2_h0(P(tc=0.0), 8193, 8.0, 20.0, 1000.0)
    k = np.nonzero(h0)[0]
    ph = np.unwrap(np.angle(h0[k]))
    tdelay = -np.diff(ph) / (2 * np.pi * (1 / 8.0))
    assert np.all(np.diff(tdelay) > 0)
    assert -1.0 < tdelay[0] < -0.7 and abs(tdelay[-1]) < 0.05      # Newtonian tau(20 Hz) = 0.962 s; 3.5PN shortens it


def test_time_domain_merger_lands_at_tc_and_chirps_up():
    # W-4: irfft of the waveform with t_c = 6 s ends (sharp band cut at f_ISCO) near 6 s
    n, fs = 16384, 2048.0
    h0 = W.taylorf2_h0(P(tc=6.0), n // 2 + 1, n / fs, 20.0, 1000.0)
    h = F.irfft(h0 * fs, n)
    e = h * h
    assert e[int(6.1 * fs):].sum() / e.sum() < 0.01
    assert e[int(5.0 * fs): int(6.1 * fs)].sum() / e.sum() > 0.5

    def zero_crossings(a):
        return np.sum(np.signbit(a[1:]) != np.signbit(a[:-1]))
    early = zero_crossings(h[int(5.0 * fs): int(5.4 * fs)])
    late = zero_crossings(h[int(5.55 * fs): int(5.95 * fs)])
    assert late > early


def test_phic_pi_symmetry_and_sign():
    a = W.taylorf2_h0(P(phic=0.4, tc=1.0), 4097, 4.0, 20.0, 1000.0)
    b = W.taylorf2_h0(P(phic=0.4 + np.pi, tc=1.0), 4097, 4.0, 20.0, 1000.0)
    assert np.abs(a - b).max() < 1e-12 * np.abs(a).max()
    c = W.taylorf2_h0(P(phic=0.4 + 0.25, tc=1.0), 4097, 4.0, 20.0, 1000.0)
    k = np.nonzero(a)[0]
    assert np.abs(c[k] / a[k] - np.exp(+2j * 0.25)).max() < 1e-9        # Psi contains -2 phi_c


def test_polarisations_face_on_edge_on():
    h0 = W.taylorf2_h0(P(), 4097, 4.0, 20.0, 1000.0)
    hp, hc = W.polarisations(h0[None], np.array([0.0]))
    assert np.allclose(np.abs(hp), np.abs(hc)) and np.allclose(hc, -1j * hp)
    hp, hc = W.polarisations(h0[None], np.array([np.pi / 2]))
    assert np.abs(hc).max() < 1e-15 * np.abs(hp).max()
    assert np.allclose(hp, 0.5 * h0)


def test_band_edges_inclusive_and_empty_band():
    # W-7: bins exactly at f_lo are kept; Mc=100,q=1 has f_ISCO=19.1 Hz < f_lo -> identically zero
    h0 = W.taylorf2_h0(P(), 4097, 4.0, 20.0, 1000.0)
    assert h0[80] != 0 and h0[79] == 0 and h0[0] == 0
    kmax = int(np.floor(W.f_isco(W.masses(26.0, 1.0)[0]) * 4.0))
    assert h0[kmax] != 0 and h0[kmax + 1] == 0
    z = W.taylorf2_h0(P(mc=100.0), 4097, 4.0, 20.0, 1000.0)
    assert np.all(z == 0) and np.all(np.isfinite(z))
    # IMR: cut at 0.2/M; Nyquist bin zero even when f_hi = fs/2
    hi = W.imrphenomd_h0(P(mc=10.0, q=1.0), 4097, 4.0, 20.0, 1024.0)
    assert hi[-1] == 0 and hi[-2] != 0


def test_invalid_parameters_give_zero_and_flag():
    bad = [P(q=1.5), P(q=0.0), P(c1=1.0), P(c2=-1.2), P(d=0.0), P(mc=-3.0)]
    for ap in (0, 1):
        hp, hc, flags = W.waveform_fd(ap, np.stack(bad + [P()]), 8192, 2048.0, 20.0, 1000.0)
        assert list(flags) == [1] * len(bad) + [0]
        assert np.all(hp[:-1] == 0) and np.all(hc[:-1] == 0) and np.any(hp[-1] != 0)


def test_optimal_snr_closed_form():
    # W-3: rho^2 = 4 A0^2 int f^(-7/3)/S df; continuum by fine trapezoid, discrete sums on the T=4, 8 s grids
    mc, q, d = 26.0, 1.0, 1000.0
    a0 = W.taylorf2_amp0(mc, d)
    fi = W.f_isco(W.masses(mc, q)[0])
    f = np.linspace(20.0, fi, 2000001)
    y = f ** (-7.0 / 3.0) / aligo_psd(f)
    rho_c = np.sqrt(4 * a0 * a0 * np.sum(0.5 * (y[1:] + y[:-1]) * np.diff(f)))
    assert abs(rho_c - G["fig1_snr_continuum"][0]) < 2e-5
    for t_seg, key in ((4.0, "fig1_snr_T4"), (8.0, "fig1_snr_T8")):
        n = int(2048 * t_seg)
        h0 = W.taylorf2_h0(P(mc=mc, q=q, d=d), n // 2 + 1, t_seg, 20.0, 1000.0)
        fk = np.arange(n // 2 + 1) / t_seg
        rho = np.sqrt(4 / t_seg * np.sum(np.abs(h0) ** 2 / aligo_psd(fk)))
        assert abs(rho - G[key][0]) < 2e-5
    h0 = W.taylorf2_h0(P(mc=10.0, q=0.25, d=200.0), 8193, 8.0, 20.0, 1000.0)
    rho = np.sqrt(4 / 8.0 * np.sum(np.abs(h0) ** 2 / aligo_psd(np.arange(8193) / 8.0)))
    assert abs(rho - G["b_snr_T8"][0]) < 2e-5


# ------------------------------- IMRPhenomD (structural pins, W-1 i..vii) -----------------

def test_table_shape():
    assert set(T.TABLE) == set(T.NAMES) and all(len(T.TABLE[k]) == 11 for k in T.NAMES)


@pytest.mark.parametrize("mc,q", [(26.0, 1.0), (10.0, 0.25), (60.0, 0.125)])
def test_imr_sigma_zero_reduces_to_taylorf2(mc, q):
    # (i) with sigma_i = 0 and chi = 0 the inspiral phase IS the TaylorF2 closed form
    mtot, eta, _, _ = W.masses(mc, q)
    pd = W.PhenomD(eta, 0.0, 0.0, sigma_scale=0.0)
    mf = np.linspace(0.002, 0.0179, 50)
    ref = W.taylorf2_phase(mf / (mtot * C.MTSUN_SI), mc, q)
    assert np.abs(pd.phi_ins(mf) - ref).max() < 1e-8 * np.abs(ref).max()


def test_pn_phase_coeffs_nonspinning_equal_published_series():
    eta = 0.2
    v, vl = W.pn_phase_coeffs(eta, 0.0, 0.0)
    assert abs(v[2] - (3715 / 756 + 55 * eta / 9)) < 1e-13
    assert abs(v[4] - (15293365 / 508032 + 27145 * eta / 504 + 3085 * eta ** 2 / 72)) < 1e-12
    assert abs(v[5] - np.pi * (38645 / 756 - 65 * eta / 9)) < 1e-12 and abs(vl[5] - 3 * v[5]) < 1e-12
    assert abs(v[7] - np.pi * (77096675 / 254016 + 378515 * eta / 1512 - 74045 * eta ** 2 / 756)) < 1e-11


@pytest.mark.parametrize("eta,c1,c2", [(0.25, 0.0, 0.0), (0.16, 0.7, -0.3), (0.0988, -0.9, 0.9),
                                       (0.2222, 0.99, 0.99), (0.25, -0.99, -0.99)])
def test_imr_c1_junctions(eta, c1, c2):
    # (ii), (iii): value and first derivative continuous at every junction (< 1e-9 rad in fp64).
    # The analytic derivative formulas used to build the junctions are themselves checked against
    # central differences of the value formulas.
    pd = W.PhenomD(eta, c1, c2)
    f1, f2 = pd.F_PHI_INS, pd.f_phi_mr
    v_int = lambda f: pd.phi_int_raw(f) + pd.c1_int + pd.c2_int * f
    v_mr = lambda f: pd.phi_mr_raw(f) + pd.c1_mr + pd.c2_mr * f
    assert abs(pd.phi_ins(f1) - v_int(f1)) < 1e-9
    assert abs(v_int(f2) - v_mr(f2)) < 1e-9
    assert abs(pd.dphi_ins(f1) - (pd.dphi_int_raw(f1) + pd.c2_int)) < 1e-9 * abs(pd.dphi_ins(f1))
    assert abs((pd.dphi_int_raw(f2) + pd.c2_int) - (pd.dphi_mr_raw(f2) + pd.c2_mr)) < 1e-9 * abs(pd.dphi_mr_raw(f2))
    e = 1e-6
    for val, der, f in ((pd.phi_ins, pd.dphi_ins, f1), (pd.phi_int_raw, pd.dphi_int_raw, f1),
                        (pd.phi_int_raw, pd.dphi_int_raw, f2), (pd.phi_mr_raw, pd.dphi_mr_raw, f2),
                        (pd.amp_ins, pd.damp_ins, pd.F_AMP_INS), (pd.amp_mr, pd.damp_mr, pd.f_peak)):
        fd = (val(f + e) - val(f - e)) / (2 * e)
        assert abs(fd - der(f)) < 1e-6 * abs(der(f)) + 1e-6 * abs(val(f)) / f
    # phase(): the assembled piecewise function has no jump across either junction
    for fj in (f1, f2):
        lo, hi = pd.phase(np.array([fj * (1 - 1e-13)]))[0], pd.phase(np.array([fj * (1 + 1e-13)]))[0]
        assert abs(hi - lo) < 1e-8
    # amplitude: value and slope of the quartic match both neighbours; v2 is hit at the midpoint
    fa, fc = pd.F_AMP_INS, pd.f_peak
    d = pd.delta
    dquart = lambda f: d[1] + 2 * d[2] * f + 3 * d[3] * f ** 2 + 4 * d[4] * f ** 3
    assert abs(pd.amp_int(fa) - pd.amp_ins(fa)) < 1e-9 and abs(pd.amp_int(fc) - pd.amp_mr(fc)) < 1e-9
    assert abs(dquart(fa) - pd.damp_ins(fa)) < 1e-7 * (1 + abs(pd.damp_ins(fa)))
    assert abs(dquart(fc) - pd.damp_mr(fc)) < 1e-7 * (1 + abs(pd.damp_mr(fc)))
    assert abs(pd.amp_int(0.5 * (fa + fc)) - pd.c["v2"]) < 1e-9
    assert np.all(pd.amplitude(np.linspace(0.001, 0.2, 2000)) > 0)
    # f_peak is where the ringdown ansatz (times f^(-7/6) removed) peaks
    # (for gamma2 > 1 the ansatz has no stationary point and [32] takes f_RD - f_damp gamma3/gamma2)
    if pd.c["gamma2"] <= 1.0:
        h = 1e-3 * pd.f_dm                       # local maximum (the other stationary point is a minimum)
        assert pd.amp_mr(fc) > pd.amp_mr(fc - h) and pd.amp_mr(fc) > pd.amp_mr(fc + h)
    else:
        assert abs(fc - abs(pd.f_rd - pd.f_dm * pd.c["gamma3"] / pd.c["gamma2"])) < 1e-15


def test_imr_low_frequency_amplitude_limit_matches_newtonian():
    # (iv): f^(7/6)|h0| -> A0 of TaylorF2 as Mf -> 1e-4 (within 1 %).  Two parts: the overall scale is
    # IDENTICAL (amp0 sqrt(2 eta/3) pi^(-1/6) (G M/c^3)^(-7/6) == A0), and the PN bracket -> 1.
    mc, q, d = 26.0, 1.0, 1000.0
    mtot, eta, _, _ = W.masses(mc, q)
    pd = W.PhenomD(eta, 0.0, 0.0)
    ms = mtot * C.MTSUN_SI
    amp0 = 2 * np.sqrt(5 / (64 * np.pi)) * mtot ** 2 * C.MTSUN_SI * C.MRSUN_SI / (d * C.MPC_SI)
    ident = amp0 * np.sqrt(2 * eta / 3) * np.pi ** (-1 / 6) * ms ** (-7.0 / 6.0)
    assert abs(ident / W.taylorf2_amp0(mc, d) - 1) < 1e-12
    assert abs(pd.amp_ins(1e-4) - 1) < 0.01
    f = 1e-4 / ms
    h0 = amp0 * pd.amplitude(np.array([1e-4]))[0]
    assert abs(h0 * f ** (7.0 / 6.0) / W.taylorf2_amp0(mc, d) - 1) < 0.01


def test_imr_exchange_symmetry_at_equal_mass():
    # (v): at q = 1 swapping chi1 <-> chi2 leaves the waveform unchanged
    a = W.imrphenomd_h0(P(c1=0.6, c2=-0.4, tc=3.0), 4097, 4.0, 20.0, 1000.0)
    b = W.imrphenomd_h0(P(c1=-0.4, c2=0.6, tc=3.0), 4097, 4.0, 20.0, 1000.0)
    assert np.abs(a - b).max() < 1e-9 * np.abs(a).max()


def test_imr_total_mass_scaling():
    # (vi): h0(f/lam; lam M, D) = lam^2 h0(f; M, D) at fixed q, chi (t_c = 0): use lam = 2 on grids T and 2T
    lam = 2.0
    a = W.imrphenomd_h0(P(mc=20.0, q=0.5, c1=0.3, c2=0.1), 2049, 2.0, 20.0, 1000.0)        # f_k = k/2
    b = W.imrphenomd_h0(P(mc=40.0, q=0.5, c1=0.3, c2=0.1), 2049, 4.0, 10.0, 500.0)         # f_k = k/4 = f/lam
    assert np.abs(b - lam ** 2 * a).max() < 1e-9 * np.abs(b).max()


def test_imr_remnant_textbook_values():
    # (vii): q = 1, chi = 0: a_f ~ 0.686, E_rad ~ 4.8 %, M f_RD ~ 0.0885, M f_damp ~ 0.0137
    assert abs(W.final_spin(0.25, 0, 0) - 0.686) < 0.007
    assert abs(W.e_rad(0.25, 0, 0) - 0.048) < 0.002
    frd, fdm = W.ringdown_freqs(0.25, 0, 0)
    assert abs(frd / 0.0885 - 1) < 0.01 and abs(fdm / 0.0137 - 1) < 0.01
    ms = 59.7323144598 * C.MTSUN_SI
    assert abs(frd / ms - 301.0) < 3.0 and abs(fdm / ms - 47.0) < 1.0
    # Schwarzschild limit of the QNM fit: M omega = 0.3737 - 0.0890 i
    f0 = (1.5251 - 1.1568) / (2 * np.pi)
    assert abs(2 * np.pi * f0 - 0.3737) < 0.006


@pytest.mark.parametrize("row", [P(tc=6.0), P(mc=10.0, q=0.125, c1=0.9, c2=-0.9, tc=6.2),
                                 P(mc=40.0, q=0.5, c1=0.5, c2=0.2, tc=6.4), P(mc=100.0, q=1.0, c1=-0.99, c2=-0.99, tc=5.7)])
def test_imr_time_domain_peak_at_tc(row):
    n, fs = 16384, 2048.0
    h0 = W.imrphenomd_h0(row, n // 2 + 1, n / fs, 20.0, 1000.0)
    assert np.all(np.isfinite(h0))
    h = F.irfft(h0 * fs, n)
    assert abs(np.argmax(np.abs(h)) / fs - row[7]) < 0.02
