"""Oracle frequency-domain waveforms (section 3.1, section 3.2).

The paper names the model (IMRPhenomD [32], whose inspiral is TaylorF2 at 3.5PN [33]) and
prints no formula.  The formulas below are the published ones of [33] (TaylorF2) and [32]
(IMRPhenomD ansatz and fit table, in oracle/phenomd_coeffs.py); DESIGN.md lists every
convention as a reading (R-W1 ... R-W11).  fp64 throughout, evaluated bin by bin on the
regular grid f_k = k / T, in the order the model is stated: masses -> PN coefficients ->
phase -> amplitude -> band cut -> polarisations.

params row layout (same as the C ABI, include/amplfi.h):
    0 mchirp [Msun]  1 q=m2/m1<=1  2 chi1  3 chi2  4 dist [Mpc]  5 theta_jn  6 phi_c
    7 t_c [s]  8 ra  9 dec  10 psi
"""
import numpy as np

from .constants import C_SI, MTSUN_SI, MRSUN_SI, MPC_SI, EULER_GAMMA
from . import phenomd_coeffs as _tab

TAYLORF2 = 0
IMRPHENOMD = 1


def masses(mchirp, q):
    """R-W8: q = m2/m1 <= 1, eta = q/(1+q)^2, M = Mc * eta^(-3/5); m1 >= m2 (solar masses)."""
    eta = q / (1.0 + q) ** 2
    mtot = mchirp * eta ** (-0.6)
    m1 = mtot / (1.0 + q)
    m2 = mtot * q / (1.0 + q)
    return mtot, eta, m1, m2


def params_valid(p):
    """include/amplfi.h: a sample with q not in (0,1], |chi|>=1, dist<=0 or mchirp<=0 is flagged
    and its waveform is identically zero."""
    mc, q, c1, c2, d = p[0], p[1], p[2], p[3], p[4]
    ok = (mc > 0) and (q > 0) and (q <= 1) and (abs(c1) < 1) and (abs(c2) < 1) and (d > 0)
    return bool(ok and np.all(np.isfinite(p)))


# ----------------------------------------------------------------------------------------
# TaylorF2, 3.5PN, non-spinning  (R-W2, R-W3; formula of ref. [33])
# ----------------------------------------------------------------------------------------

def taylorf2_phase(f, mchirp, q, t_c=0.0, phi_c=0.0):
    """Psi(f) = 2 pi f t_c - 2 phi_c - pi/4 + 3/(128 eta v^5) sum_j p_j v^j,  v = (pi M f)^(1/3)."""
    f = np.asarray(f, dtype=np.float64)
    mtot, eta, _, _ = masses(mchirp, q)
    ms = mtot * MTSUN_SI
    v = np.cbrt(np.pi * ms * f)
    pi = np.pi
    p0 = 1.0
    p2 = 3715.0 / 756.0 + 55.0 * eta / 9.0
    p3 = -16.0 * pi
    p4 = 15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta ** 2 / 72.0
    p5 = pi * (38645.0 / 756.0 - 65.0 * eta / 9.0) * (1.0 + 3.0 * np.log(v))
    p6 = (11583231236531.0 / 4694215680.0 - 640.0 * pi ** 2 / 3.0 - 6848.0 * EULER_GAMMA / 21.0
          + eta * (-15737765635.0 / 3048192.0 + 2255.0 * pi ** 2 / 12.0)
          + 76055.0 * eta ** 2 / 1728.0 - 127825.0 * eta ** 3 / 1296.0
          - (6848.0 / 21.0) * np.log(4.0 * v))
    p7 = pi * (77096675.0 / 254016.0 + 378515.0 * eta / 1512.0 - 74045.0 * eta ** 2 / 756.0)
    series = p0 + p2 * v ** 2 + p3 * v ** 3 + p4 * v ** 4 + p5 * v ** 5 + p6 * v ** 6 + p7 * v ** 7
    return 2.0 * pi * f * t_c - 2.0 * phi_c - pi / 4.0 + 3.0 / (128.0 * eta * v ** 5) * series


def taylorf2_amp0(mchirp, dist_mpc):
    """R-W3: A0 = sqrt(5/24) pi^(-2/3) (G Mc/c^3)^(5/6) c / D   [|h0(f)| = A0 f^(-7/6)]."""
    return np.sqrt(5.0 / 24.0) * np.pi ** (-2.0 / 3.0) * (mchirp * MTSUN_SI) ** (5.0 / 6.0) \
        * C_SI / (dist_mpc * MPC_SI)


def f_isco(mtot):
    """f_ISCO = c^3 / (6^(3/2) pi G M)."""
    return 1.0 / (6.0 ** 1.5 * np.pi * mtot * MTSUN_SI)


def chirp_time(f, mchirp):
    """Newtonian chirp time tau(f) = (5/256) (pi f)^(-8/3) (G Mc/c^3)^(-5/3)."""
    return 5.0 / 256.0 * (np.pi * f) ** (-8.0 / 3.0) * (mchirp * MTSUN_SI) ** (-5.0 / 3.0)


def taylorf2_h0(p, n_bins, t_seg, f_lo, f_hi):
    """Common complex factor h0(f_k) = A0 f^(-7/6) exp(-i Psi) on f_lo <= f_k <= min(f_ISCO, f_hi),
    zero elsewhere; DC and the last (Nyquist) bin are always zero (R-W7)."""
    h0 = np.zeros(n_bins, dtype=np.complex128)
    if not params_valid(p):
        return h0
    mchirp, q, dist, phi_c, t_c = p[0], p[1], p[4], p[6], p[7]
    mtot, _, _, _ = masses(mchirp, q)
    f_top = min(f_isco(mtot), f_hi)
    k = np.arange(n_bins)
    f = k / t_seg
    band = (f >= f_lo) & (f <= f_top) & (k > 0) & (k < n_bins - 1)
    fb = f[band]
    psi = taylorf2_phase(fb, mchirp, q, t_c, phi_c)
    h0[band] = taylorf2_amp0(mchirp, dist) * fb ** (-7.0 / 6.0) * np.exp(-1j * psi)
    return h0


# ----------------------------------------------------------------------------------------
# IMRPhenomD  (R-W1, R-W11; ansatz and fits of ref. [32])
# ----------------------------------------------------------------------------------------

def final_spin(eta, chi1, chi2):
    """Remnant spin fit used by [32] (its eq. 3.6); s = m1^2 chi1 + m2^2 chi2 with m1+m2 = 1."""
    seta = np.sqrt(max(1.0 - 4.0 * eta, 0.0))
    m1 = 0.5 * (1.0 + seta)
    m2 = 0.5 * (1.0 - seta)
    s = m1 * m1 * chi1 + m2 * m2 * chi2
    e2, e3, e4 = eta ** 2, eta ** 3, eta ** 4
    return (3.4641016151377544 * eta - 4.399247300629289 * e2 + 9.397292189321194 * e3
            - 13.180949901606242 * e4
            + (1.0 - 0.0850917821418767 * eta - 5.837029316602263 * e2) * s
            + (0.1014665242971878 * eta - 2.0967746996832157 * e2) * s ** 2
            + (-1.3546806617824356 * eta + 4.108962025369336 * e2) * s ** 3
            + (-0.8676969352555539 * eta + 2.064046835273906 * e2) * s ** 4)


def e_rad(eta, chi1, chi2):
    """Radiated-energy fit used by [32] (its eq. 3.7/3.8)."""
    seta = np.sqrt(max(1.0 - 4.0 * eta, 0.0))
    m1 = 0.5 * (1.0 + seta)
    m2 = 0.5 * (1.0 - seta)
    s = (m1 * m1 * chi1 + m2 * m2 * chi2) / (m1 * m1 + m2 * m2)
    e2, e3 = eta ** 2, eta ** 3
    return (eta * (0.055974469826360077 + 0.5809510763115132 * eta - 0.9606726679372312 * e2
                   + 3.352411249771192 * e3)
            * (1.0 + (-0.0030302335878845507 - 2.0066110851351073 * eta + 7.7050567802399215 * e2) * s)
            ) / (1.0 + (-0.6714403054720589 - 1.4756929437702908 * eta + 7.304676214885011 * e2) * s)


def ringdown_freqs(eta, chi1, chi2):
    """(M f_RD, M f_damp) of the l = m = 2, n = 0 Kerr mode of the remnant, in units of the INITIAL total mass:
    f_RD = Re(omega)/(2 pi), f_damp = -Im(omega)/(2 pi) with M_f omega of the mode at the final spin (oracle/qnm.py:
    Leaver's continued fractions, tabulated and spline-interpolated, i.e. the function whose Berti-Cardoso-Will
    tabulation [32] interpolates), both divided by the remnant mass 1 - E_rad.  Reading R-W1b."""
    from .qnm import qnm_220
    a = final_spin(eta, chi1, chi2)
    w_re, w_im = qnm_220(a)
    m_f = 1.0 - e_rad(eta, chi1, chi2)
    return w_re / (2.0 * np.pi) / m_f, w_im / (2.0 * np.pi) / m_f


def ringdown_freqs_fit(eta, chi1, chi2):
    """The same from the Berti-Cardoso-Will closed-form fit (f = [1.5251 - 1.1568 (1-a)^0.1292]/(2 pi),
    Q = 0.7 + 1.4187 (1-a)^(-0.4990), f_damp = f/(2Q); accurate to a few per cent): kept as a cross-check of the table."""
    a = final_spin(eta, chi1, chi2)
    a = min(max(a, -0.999999), 0.999999)
    f_ring = (1.5251 - 1.1568 * (1.0 - a) ** 0.1292) / (2.0 * np.pi)
    qual = 0.7 + 1.4187 * (1.0 - a) ** (-0.4990)
    f_damp = f_ring / (2.0 * qual)
    m_f = 1.0 - e_rad(eta, chi1, chi2)
    return f_ring / m_f, f_damp / m_f


def chi_pn(eta, chi1, chi2):
    """chi_PN = chi_eff - (38 eta / 113)(chi1 + chi2), chi_eff = (m1 chi1 + m2 chi2)/M  ([32] eq. 1.5)."""
    seta = np.sqrt(max(1.0 - 4.0 * eta, 0.0))
    m1 = 0.5 * (1.0 + seta)
    m2 = 0.5 * (1.0 - seta)
    return m1 * chi1 + m2 * chi2 - 38.0 * eta / 113.0 * (chi1 + chi2)


def pn_phase_coeffs(eta, chi1, chi2):
    """TaylorF2 aligned-spin phasing series used as the IMRPhenomD inspiral ([32] App. B; [33]).

    Returns (v, vlogv): phase = 3/(128 eta) * sum_i (v[i] + vlogv[i] ln v) v^(i-5).
    Spin terms: spin-orbit at 1.5, 2.5, 3 (tail) and 3.5PN, spin-spin at 2PN (black-hole
    quadrupole); the 3PN spin-spin term is NOT included (as in [32]).  chi = 0 reduces to
    taylorf2_phase exactly.
    """
    pi = np.pi
    seta = np.sqrt(max(1.0 - 4.0 * eta, 0.0))
    m1 = 0.5 * (1.0 + seta)
    m2 = 0.5 * (1.0 - seta)
    d = m1 - m2
    sl = m1 * m1 * chi1 + m2 * m2 * chi2
    dsl = d * (m2 * chi2 - m1 * chi1)
    v = np.zeros(8)
    vl = np.zeros(8)
    v[0] = 1.0
    v[2] = 5.0 * (743.0 / 84.0 + 11.0 * eta) / 9.0
    v[3] = -16.0 * pi
    v[4] = 5.0 * (3058.673 / 7.056 + 5429.0 / 7.0 * eta + 617.0 * eta * eta) / 72.0
    v[5] = 5.0 / 9.0 * (7729.0 / 84.0 - 13.0 * eta) * pi
    vl[5] = 5.0 / 3.0 * (7729.0 / 84.0 - 13.0 * eta) * pi
    v[6] = (11583.231236531 / 4.694215680 - 640.0 / 3.0 * pi * pi - 6848.0 / 21.0 * EULER_GAMMA
            + eta * (-15737.765635 / 3.048192 + 2255.0 / 12.0 * pi * pi)
            + eta * eta * 76055.0 / 1728.0 - eta ** 3 * 127825.0 / 1296.0
            - 6848.0 / 21.0 * np.log(4.0))
    vl[6] = -6848.0 / 21.0
    v[7] = pi * (77096675.0 / 254016.0 + 378515.0 / 1512.0 * eta - 74045.0 / 756.0 * eta * eta)
    # spin-orbit 3.5PN
    v[7] += ((-8980424995.0 / 762048.0 + 6586595.0 * eta / 756.0 - 305.0 * eta * eta / 36.0) * sl
             - (170978035.0 / 48384.0 - 2876425.0 * eta / 672.0 - 4735.0 * eta * eta / 144.0) * dsl)
    # spin-orbit 3PN (tail)
    v[6] += pi * (3760.0 * sl + 1490.0 * dsl) / 3.0
    # spin-orbit 2.5PN
    gam = (554345.0 / 1134.0 + 110.0 * eta / 9.0) * sl + (13915.0 / 84.0 - 10.0 * eta / 3.0) * dsl
    v[5] += -gam
    vl[5] += -3.0 * gam
    # spin-spin 2PN (aligned spins, quadrupole-monopole of a black hole)
    sig = eta * (721.0 / 48.0 - 247.0 / 48.0) * chi1 * chi2
    sig += (719.0 / 96.0 - 233.0 / 96.0) * (m1 * m1 * chi1 * chi1 + m2 * m2 * chi2 * chi2)
    v[4] += -10.0 * sig
    # spin-orbit 1.5PN
    v[3] += 188.0 * sl / 3.0 + 25.0 * dsl
    return v, vl


def amp_pn_coeffs(eta, chi1, chi2):
    """Coefficients A_2..A_6 of the PN-expanded inspiral amplitude in powers of (pi M f)^(i/3)
    ([32] eq. 29 and App. B)."""
    pi = np.pi
    seta = np.sqrt(max(1.0 - 4.0 * eta, 0.0))
    e2, e3 = eta * eta, eta ** 3
    c12, c22 = chi1 * chi1, chi2 * chi2
    a2 = (-969.0 + 1804.0 * eta) / 672.0
    a3 = (chi1 * (81.0 * (1.0 + seta) - 44.0 * eta) + chi2 * (81.0 - 81.0 * seta - 44.0 * eta)) / 48.0
    a4 = (-27312085.0 - 10287648.0 * c22 - 10287648.0 * c12 * (1.0 + seta) + 10287648.0 * c22 * seta
          + 24.0 * (-1975055.0 + 857304.0 * c12 - 994896.0 * chi1 * chi2 + 857304.0 * c22) * eta
          + 35371056.0 * e2) / 8128512.0
    a5 = (chi2 * (-285197.0 * (-1.0 + seta) + 4.0 * (-91902.0 + 1579.0 * seta) * eta - 35632.0 * e2)
          + chi1 * (285197.0 * (1.0 + seta) - 4.0 * (91902.0 + 1579.0 * seta) * eta - 35632.0 * e2)
          + 42840.0 * (-1.0 + 4.0 * eta) * pi) / 32256.0
    a6 = -(-336.0 * (-3248849057.0 + 2943675504.0 * c12 - 3339284256.0 * chi1 * chi2
                     + 2943675504.0 * c22) * e2
           - 324322727232.0 * e3
           - 7.0 * (-177520268561.0 + 107414046432.0 * c22 + 107414046432.0 * c12 * (1.0 + seta)
                    - 107414046432.0 * c22 * seta
                    + 11087290368.0 * (chi1 + chi2 + chi1 * seta - chi2 * seta) * pi)
           + 12.0 * eta * (-545384828789.0 - 176491177632.0 * chi1 * chi2 + 202603761360.0 * c22
                           + 77616.0 * c12 * (2610335.0 + 995766.0 * seta)
                           - 77287373856.0 * c22 * seta
                           + 5841690624.0 * (chi1 + chi2) * pi + 21384760320.0 * pi * pi)
           ) / 60085960704.0
    return a2, a3, a4, a5, a6


class PhenomD:
    """All per-sample quantities of IMRPhenomD for (eta, chi1, chi2), geometric units (Mf).

    Follows [32] in its own order: fit coefficients -> ringdown -> inspiral phase -> C1 junctions
    at Mf = 0.018 and 0.5 f_RD -> amplitude regions with junctions at Mf = 0.014 and f_peak.
    ``sigma_scale`` / ``tab`` exist for the structural pins (sigma = 0 must give TaylorF2).
    """
    F_PHI_INS = 0.018
    F_AMP_INS = 0.014
    F_CUT = 0.2

    def __init__(self, eta, chi1, chi2, tab=None, sigma_scale=1.0):
        tab = _tab.TABLE if tab is None else tab
        self.eta, self.chi1, self.chi2 = eta, chi1, chi2
        xi = chi_pn(eta, chi1, chi2) - 1.0
        c = {name: _tab.evaluate(tab[name], eta, xi) for name in _tab.NAMES}
        for s in ("sigma1", "sigma2", "sigma3", "sigma4"):
            c[s] *= sigma_scale
        self.c = c
        self.f_rd, self.f_dm = ringdown_freqs(eta, chi1, chi2)
        self.v, self.vl = pn_phase_coeffs(eta, chi1, chi2)
        self.amp_a = amp_pn_coeffs(eta, chi1, chi2)
        # ---- phase junctions (C1) ----
        f1 = self.F_PHI_INS
        f2 = 0.5 * self.f_rd
        self.f_phi_mr = f2
        self.c2_int = self.dphi_ins(f1) - self.dphi_int_raw(f1)
        self.c1_int = self.phi_ins(f1) - self.phi_int_raw(f1) - self.c2_int * f1
        self.c2_mr = (self.dphi_int_raw(f2) + self.c2_int) - self.dphi_mr_raw(f2)
        self.c1_mr = (self.phi_int_raw(f2) + self.c1_int + self.c2_int * f2) \
            - self.phi_mr_raw(f2) - self.c2_mr * f2
        # ---- amplitude: peak frequency and intermediate quartic ----
        g2, g3 = c["gamma2"], c["gamma3"]
        if g2 > 1.0:
            self.f_peak = abs(self.f_rd - self.f_dm * g3 / g2)
        else:
            self.f_peak = abs(self.f_rd + self.f_dm * (np.sqrt(1.0 - g2 * g2) - 1.0) * g3 / g2)
        fa, fc = self.F_AMP_INS, self.f_peak
        fb = 0.5 * (fa + fc)
        rows = [[1.0, fa, fa ** 2, fa ** 3, fa ** 4],
                [1.0, fb, fb ** 2, fb ** 3, fb ** 4],
                [1.0, fc, fc ** 2, fc ** 3, fc ** 4],
                [0.0, 1.0, 2 * fa, 3 * fa ** 2, 4 * fa ** 3],
                [0.0, 1.0, 2 * fc, 3 * fc ** 2, 4 * fc ** 3]]
        rhs = [self.amp_ins(fa), c["v2"], self.amp_mr(fc), self.damp_ins(fa), self.damp_mr(fc)]
        self.delta = np.linalg.solve(np.array(rows), np.array(rhs))
        # ---- time alignment: slope of the merger-ringdown phase at the amplitude peak ----
        self.t0 = self.dphi_mr_raw(self.f_peak) + self.c2_mr

    # ---------------- phase ----------------
    def phi_ins(self, f):
        eta, c = self.eta, self.c
        v = np.cbrt(np.pi * f)
        lv = np.log(v)
        tf2 = sum((self.v[i] + self.vl[i] * lv) * v ** (i - 5) for i in range(8))
        tf2 = 3.0 / (128.0 * eta) * tf2 - np.pi / 4.0
        return tf2 + (c["sigma1"] * f + 0.75 * c["sigma2"] * f ** (4.0 / 3.0)
                      + 0.6 * c["sigma3"] * f ** (5.0 / 3.0) + 0.5 * c["sigma4"] * f ** 2) / eta

    def dphi_ins(self, f):
        """d phi_ins / d(Mf), term by term."""
        eta, c = self.eta, self.c
        v = np.cbrt(np.pi * f)
        lv = np.log(v)
        dv = v / (3.0 * f)                                         # dv/df
        s = sum(((i - 5) * (self.v[i] + self.vl[i] * lv) + self.vl[i]) * v ** (i - 6) for i in range(8))
        return 3.0 / (128.0 * eta) * s * dv + (c["sigma1"] + c["sigma2"] * f ** (1.0 / 3.0)
                                               + c["sigma3"] * f ** (2.0 / 3.0) + c["sigma4"] * f) / eta

    def phi_int_raw(self, f):
        c = self.c
        return (c["beta1"] * f + c["beta2"] * np.log(f) - c["beta3"] / (3.0 * f ** 3)) / self.eta

    def dphi_int_raw(self, f):
        c = self.c
        return (c["beta1"] + c["beta2"] / f + c["beta3"] / f ** 4) / self.eta

    def phi_mr_raw(self, f):
        c = self.c
        return (c["alpha1"] * f - c["alpha2"] / f + 4.0 / 3.0 * c["alpha3"] * f ** 0.75
                + c["alpha4"] * np.arctan((f - c["alpha5"] * self.f_rd) / self.f_dm)) / self.eta

    def dphi_mr_raw(self, f):
        c = self.c
        x = (f - c["alpha5"] * self.f_rd) / self.f_dm
        return (c["alpha1"] + c["alpha2"] / f ** 2 + c["alpha3"] * f ** (-0.25)
                + c["alpha4"] / (self.f_dm * (1.0 + x * x))) / self.eta

    def phase(self, f):
        """phi_IMR(Mf): the three regions joined C1."""
        f = np.asarray(f, dtype=np.float64)
        out = np.empty_like(f)
        r1 = f < self.F_PHI_INS
        r3 = f >= self.f_phi_mr
        r2 = ~(r1 | r3)
        out[r1] = self.phi_ins(f[r1])
        out[r2] = self.phi_int_raw(f[r2]) + self.c1_int + self.c2_int * f[r2]
        out[r3] = self.phi_mr_raw(f[r3]) + self.c1_mr + self.c2_mr * f[r3]
        return out

    # ---------------- amplitude (all regions multiply amp0' * f^(-7/6)) ----------------
    def amp_ins(self, f):
        a2, a3, a4, a5, a6 = self.amp_a
        c = self.c
        x = np.cbrt(np.pi * f)
        return (1.0 + a2 * x ** 2 + a3 * x ** 3 + a4 * x ** 4 + a5 * x ** 5 + a6 * x ** 6
                + c["rho1"] * f ** (7.0 / 3.0) + c["rho2"] * f ** (8.0 / 3.0) + c["rho3"] * f ** 3)

    def damp_ins(self, f):
        a2, a3, a4, a5, a6 = self.amp_a
        c = self.c
        x = np.cbrt(np.pi * f)
        dx = x / (3.0 * f)
        return ((2 * a2 * x + 3 * a3 * x ** 2 + 4 * a4 * x ** 3 + 5 * a5 * x ** 4 + 6 * a6 * x ** 5) * dx
                + 7.0 / 3.0 * c["rho1"] * f ** (4.0 / 3.0) + 8.0 / 3.0 * c["rho2"] * f ** (5.0 / 3.0)
                + 3.0 * c["rho3"] * f ** 2)

    def amp_mr(self, f):
        c = self.c
        w = self.f_dm * c["gamma3"]
        return np.exp(-(f - self.f_rd) * c["gamma2"] / w) * (w * c["gamma1"]) / ((f - self.f_rd) ** 2 + w * w)

    def damp_mr(self, f):
        c = self.c
        w = self.f_dm * c["gamma3"]
        d = f - self.f_rd
        lor = (w * c["gamma1"]) / (d * d + w * w)
        ex = np.exp(-d * c["gamma2"] / w)
        return ex * lor * (-c["gamma2"] / w - 2.0 * d / (d * d + w * w))

    def amp_int(self, f):
        d = self.delta
        return d[0] + f * (d[1] + f * (d[2] + f * (d[3] + f * d[4])))

    def amplitude(self, f):
        """A(Mf) without the overall strain scale: sqrt(2 eta/3) pi^(-1/6) f^(-7/6) * region."""
        f = np.asarray(f, dtype=np.float64)
        out = np.empty_like(f)
        r1 = f < self.F_AMP_INS
        r3 = f >= self.f_peak
        r2 = ~(r1 | r3)
        out[r1] = self.amp_ins(f[r1])
        out[r2] = self.amp_int(f[r2])
        out[r3] = self.amp_mr(f[r3])
        return np.sqrt(2.0 * self.eta / 3.0) * np.pi ** (-1.0 / 6.0) * f ** (-7.0 / 6.0) * out


def imrphenomd_h0(p, n_bins, t_seg, f_lo, f_hi, tab=None, sigma_scale=1.0):
    """h0(f_k) = amp0 * A(Mf) * exp(-i Psi),  Psi = 2 pi f t_c - 2 phi_c + phi_IMR(Mf) - t0 * Mf
    on f_lo <= f_k <= min(0.2/M, f_hi); zero elsewhere, DC and Nyquist always zero (R-W7).
    amp0 = 2 sqrt(5/(64 pi)) M^2 (G Msun/c^3)(G Msun/c^2) / D.  t0 puts the amplitude peak at t_c."""
    h0 = np.zeros(n_bins, dtype=np.complex128)
    if not params_valid(p):
        return h0
    mchirp, q, chi1, chi2, dist, phi_c, t_c = p[0], p[1], p[2], p[3], p[4], p[6], p[7]
    mtot, eta, _, _ = masses(mchirp, q)
    ms = mtot * MTSUN_SI
    pd = PhenomD(eta, chi1, chi2, tab=tab, sigma_scale=sigma_scale)
    f_top = min(PhenomD.F_CUT / ms, f_hi)
    k = np.arange(n_bins)
    f = k / t_seg
    band = (f >= f_lo) & (f <= f_top) & (k > 0) & (k < n_bins - 1)
    fb = f[band]
    mf = ms * fb
    amp0 = 2.0 * np.sqrt(5.0 / (64.0 * np.pi)) * mtot * mtot * MTSUN_SI * MRSUN_SI / (dist * MPC_SI)
    psi = 2.0 * np.pi * fb * t_c - 2.0 * phi_c + pd.phase(mf) - pd.t0 * mf
    h0[band] = amp0 * pd.amplitude(mf) * np.exp(-1j * psi)
    return h0


# ----------------------------------------------------------------------------------------
# Sine-Gaussian burst ("can be extended to burst signal morphologies like sine-Gaussians ...
# central frequency or duration").  The paper gives no formula: DESIGN.md reading R-W12.
# ----------------------------------------------------------------------------------------
SINE_GAUSSIAN = 2


def sg_params_valid(p):
    """row layout for this family: 0 f0 [Hz], 1 Q, 2-3 unused, 4 peak amplitude A, 5 ellipticity angle iota,
    6 phase phi, 7 central time t0 [s], 8 ra, 9 dec, 10 psi."""
    return bool((p[0] > 0) and (p[1] > 0) and (p[4] > 0) and np.all(np.isfinite(p)))


def sine_gaussian_td(p, t):
    """Time-domain definition: h+(t) = (1 + cos^2 iota)/2 * A e^{-(t-t0)^2/tau^2} cos(2 pi f0 (t-t0) + phi),
    hx(t) = cos iota * A e^{-(t-t0)^2/tau^2} sin(2 pi f0 (t-t0) + phi),  tau = Q / (sqrt 2 pi f0)."""
    f0, q, amp, iota, phi, t0 = p[0], p[1], p[4], p[5], p[6], p[7]
    tau = q / (np.sqrt(2.0) * np.pi * f0)
    env = amp * np.exp(-((t - t0) / tau) ** 2)
    arg = 2.0 * np.pi * f0 * (t - t0) + phi
    ci = np.cos(iota)
    return 0.5 * (1.0 + ci * ci) * env * np.cos(arg), ci * env * np.sin(arg)


def sine_gaussian_h0(p, n_bins, t_seg, f_lo, f_hi):
    """Frequency-domain model on the grid, positive-frequency Gaussian only (the mirror term centred on -f0 is dropped:
    it is e^{-2 Q^2} of the peak at f0 and at most e^{-Q^2/2} of it anywhere, reached as f -> 0): h0(f) = A tau sqrt(pi)/2 * e^{-pi^2 tau^2 (f - f0)^2} * e^{-i (2 pi f t0 - phi)},
    with h+ = (1 + cos^2 iota)/2 h0 and hx = -i cos iota h0 as for the binaries (R-W6); non-zero for
    f_lo <= f_k <= f_hi, bins 0 and Nyquist always zero (R-W7)."""
    h0 = np.zeros(n_bins, dtype=np.complex128)
    if not sg_params_valid(p):
        return h0
    f0, q, amp, phi, t0 = p[0], p[1], p[4], p[6], p[7]
    tau = q / (np.sqrt(2.0) * np.pi * f0)
    k = np.arange(n_bins)
    f = k / t_seg
    band = (f >= f_lo) & (f <= f_hi) & (k > 0) & (k < n_bins - 1)
    fb = f[band]
    h0[band] = 0.5 * amp * tau * np.sqrt(np.pi) * np.exp(-(np.pi * tau * (fb - f0)) ** 2) \
        * np.exp(-1j * (2.0 * np.pi * fb * t0 - phi))
    return h0


# ----------------------------------------------------------------------------------------
# batch entry point mirroring amplfi_waveform_fd
# ----------------------------------------------------------------------------------------

def h0_fd(approximant, params, n, fs, f_lo, f_hi):
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    n_bins = n // 2 + 1
    t_seg = n / fs
    fn = {TAYLORF2: taylorf2_h0, IMRPHENOMD: imrphenomd_h0, SINE_GAUSSIAN: sine_gaussian_h0}[approximant]
    return np.stack([fn(p, n_bins, t_seg, f_lo, f_hi) for p in params])


def polarisations(h0, theta_jn):
    """R-W6: iota = theta_JN; h+ = (1 + cos^2 iota)/2 * h0,  hx = -i cos iota * h0."""
    ci = np.cos(np.asarray(theta_jn, dtype=np.float64))[..., None]
    return 0.5 * (1.0 + ci * ci) * h0, -1j * ci * h0


def waveform_fd(approximant, params, n, fs, f_lo, f_hi):
    """Returns (hp, hc, flags): [B, K] complex128 each, flags[b] = 1 for an invalid sample."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    h0 = h0_fd(approximant, params, n, fs, f_lo, f_hi)
    hp, hc = polarisations(h0, params[:, 5])
    valid = sg_params_valid if approximant == SINE_GAUSSIAN else params_valid
    flags = np.array([0 if valid(p) else 1 for p in params], dtype=np.int32)
    return hp, hc, flags


def waveform_td(approximant, params, n, fs, f_lo, f_hi):
    """Time-domain polarisations on the segment grid t_j = j/fs (Figure 1 compares the
    "time-domain IMRPhenomD").  The frequency-domain model is the definition; its time series is
    the inverse Fourier integral sampled on the grid, h(t_j) = df * sum over the two-sided spectrum of
    h~(f_k) exp(+2 pi i f_k t_j) = fs * irfft(h~)[j]  (circular on the segment: reading R-W9).
    Returns (hp_t, hc_t, flags): [B, n] float64 each."""
    from .fft import irfft
    hp, hc, flags = waveform_fd(approximant, params, n, fs, f_lo, f_hi)
    return fs * irfft(hp, n), fs * irfft(hc, n), flags
