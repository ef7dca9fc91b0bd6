"""Pins for oracle.qnm: the Kerr (2,2,0) quasi-normal mode that sets the ringdown of IMRPhenomD ([32])."""
import numpy as np
import pytest

from oracle import qnm
from oracle import waveform as W


def test_schwarzschild_and_published_kerr_values():
    """Leaver (1985) Table 1 / Berti, Cardoso & Starinets (2009): M omega of the l = m = 2 fundamental mode."""
    w0, sep0 = qnm.kerr_qnm_220(0.0)
    assert abs(w0 - (0.37367168 - 0.08896232j)) < 2e-8
    assert abs(sep0 - 4.0) < 1e-10                       # A_lm = l(l+1) - s(s+1) at a = 0
    s, wr, wi = qnm.ringdown_table()
    for spin, ref in ((0.7, 0.5326 - 0.0808j), (0.9, 0.6716 - 0.0649j)):
        i = int(np.argmin(np.abs(s - spin)))
        w, _ = qnm.kerr_qnm_220(spin, start=(s[i], wr[i] - 1j * wi[i], _sep_guess(s[i])))
        assert abs(w - ref) < 6e-5


def _sep_guess(spin):
    # separation constant of the spin-weighted spheroidal harmonic to second order in a omega (enough for a starting guess)
    return 4.0 - 2.0 * spin * 0.5 * 8.0 / 6.0


def test_table_nodes_are_solutions_of_the_continued_fractions():
    s, wr, wi = qnm.ringdown_table()
    assert len(s) == 401 and np.all(np.diff(s) > 0) and s[0] == pytest.approx(-0.998) and s[-1] == pytest.approx(0.998)
    w, sep = qnm.kerr_qnm_220(s[260])                    # an independent walk from Schwarzschild
    assert abs(w.real - wr[260]) < 1e-10 and abs(-w.imag - wi[260]) < 1e-10
    for i, j in ((0, 12), (57, 70), (333, 320), (400, 392)):
        # re-solved from the solution at a node a few steps away (the separation constant from a short walk there)
        _, sep_j = qnm.kerr_qnm_220(s[j], start=(s[260], w, sep)) if abs(s[j] - s[260]) < 0.3 else qnm.kerr_qnm_220(s[j])
        wi_, sep_i = qnm.kerr_qnm_220(s[i], start=(s[j], wr[j] - 1j * wi[j], sep_j))
        assert abs(wi_.real - wr[i]) < 1e-10 and abs(-wi_.imag - wi[i]) < 1e-10
        f_ang, f_rad = qnm.leaver_conditions(2.0 * wi_, sep_i, 0.5 * s[i])
        assert abs(f_ang) < 1e-8 and abs(f_rad) < 1e-8


def test_spline_between_nodes_and_monotone_trends():
    s, wr, wi = qnm.ringdown_table()
    mid = 0.5 * (s[250] + s[251])
    w, _ = qnm.kerr_qnm_220(mid)
    r, i = qnm.qnm_220(mid)
    assert abs(w.real - r) < 1e-9 and abs(-w.imag - i) < 1e-9
    assert np.all(np.diff(wr) > 0)                        # the frequency rises with the spin,
    assert np.all(np.diff(wi[s > 0.0]) < 0)               # the damping falls for co-rotating modes,
    assert wr[-1] < 1.0 and wi[-1] > 0.0                  # towards M omega -> m/2 = 1, Im -> 0 at the extremal hole


def test_berti_cardoso_will_fit_agrees_within_its_accuracy():
    """The closed-form fit the first round used (and lalsimulation's data it approximates) is good to a few per cent."""
    for a in np.linspace(0.0, 0.95, 20):                  # (the fit was made for co-rotating modes)
        wr, wi = qnm.qnm_220(a)
        f_fit = 1.5251 - 1.1568 * (1.0 - a) ** 0.1292
        q_fit = 0.7 + 1.4187 * (1.0 - a) ** (-0.4990)
        assert abs(f_fit / wr - 1.0) < 0.03
        assert abs(q_fit / (wr / (2.0 * wi)) - 1.0) < 0.06
    frd, fdm = W.ringdown_freqs(0.25, 0.0, 0.0)
    frd2, fdm2 = W.ringdown_freqs_fit(0.25, 0.0, 0.0)
    assert abs(frd / frd2 - 1) < 0.02 and abs(fdm / fdm2 - 1) < 0.03
