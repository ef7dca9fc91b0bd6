"""Oracle: the l = m = 2, n = 0 quasi-normal mode of a Kerr black hole (test infrastructure).

IMRPhenomD [32] takes its ringdown frequency and damping time from the tabulated Kerr QNM data of
Berti, Cardoso & Will; that table is a tabulation of a function mathematics defines: the frequency at which the
Teukolsky equation (spin weight s = -2) has a solution that is ingoing at the horizon and outgoing at infinity.
Leaver's method (Proc. R. Soc. A 402, 285 (1985)) turns both the angular and the radial equation into three-term
recurrences whose continued fractions must vanish; the two conditions are solved here for (omega, A_lm) by Newton
iteration, continued in the spin from the Schwarzschild value.  Units G = c = 1 and, as in Leaver's paper, 2 M = 1
inside the recurrences; the public functions take the dimensionless spin a/M in (-1, 1) (negative: the mode that
counter-rotates with the hole) and return M omega.

``kerr_qnm_220`` solves directly (slow: tens of ms per spin); ``ringdown_table`` reads oracle/qnm_220_table.txt, written by
oracle/make_qnm_table.py from this solver, and ``qnm_220`` interpolates it with a cubic spline (what oracle.waveform uses).
Pins: tests/test_oracle_qnm.py (Schwarzschild 0.37367 - 0.08896 i, the published a/M = 0.7 and 0.9 values, the
Berti-Cardoso-Will fit within its stated accuracy, the extremal limit, table nodes against direct solves).
"""
import os

import numpy as np

S, L, M_AZ = -2, 2, 2


def _continued_fraction(alpha, beta, gamma, depth):
    """beta_0 - alpha_0 gamma_1 / (beta_1 - alpha_1 gamma_2 / (beta_2 - ...)), evaluated bottom-up from `depth`."""
    t = 0.0
    for n in range(depth, 0, -1):
        t = alpha(n - 1) * gamma(n) / (beta(n) - t)
    return beta(0) - t


def leaver_conditions(w, sep, a, depth_radial=3000, depth_angular=120):
    """The two continued-fraction conditions (angular, radial) at frequency w, separation constant sep, spin a (2M = 1)."""
    b = np.sqrt(1.0 - 4.0 * a * a)
    k1 = 0.5 * abs(M_AZ - S)
    k2 = 0.5 * abs(M_AZ + S)

    def a_al(n):
        return -2.0 * (n + 1) * (n + 2 * k1 + 1)

    def a_be(n):
        return (n * (n - 1) + 2 * n * (k1 + k2 + 1 - 2 * a * w)
                - (2 * a * w * (2 * k1 + S + 1) - (k1 + k2) * (k1 + k2 + 1)) - (a * a * w * w + S * (S + 1) + sep))

    def a_ga(n):
        return 2 * a * w * (n + k1 + k2 + S)

    q = 0.5 * w - a * M_AZ
    c0 = 1 - S - 1j * w - (2j / b) * q
    c1 = -4 + 2j * w * (2 + b) + (4j / b) * q
    c2 = S + 3 - 3j * w - (2j / b) * q
    c3 = w * w * (4 + 2 * b - a * a) - 2 * a * M_AZ * w - S - 1 + (2 + b) * 1j * w - sep + ((4 * w + 2j) / b) * q
    c4 = S + 1 - 2 * w * w - (2 * S + 3) * 1j * w - ((4 * w + 2j) / b) * q

    def r_al(n):
        return n * n + (c0 + 1) * n + c0

    def r_be(n):
        return -2 * n * n + (c1 + 2) * n + c3

    def r_ga(n):
        return n * n + (c2 - 3) * n + c4 - c2 + 2

    return (_continued_fraction(a_al, a_be, a_ga, depth_angular),
            _continued_fraction(r_al, r_be, r_ga, depth_radial))


def _newton(a, w, sep, tol=1e-13, max_iter=40):
    """Newton iteration on the two complex conditions in the two complex unknowns (finite-difference Jacobian)."""
    for _ in range(max_iter):
        f0 = np.array(leaver_conditions(w, sep, a))
        h = 1e-7
        fw = np.array(leaver_conditions(w + h, sep, a))
        fs = np.array(leaver_conditions(w, sep + h, a))
        jac = np.column_stack([(fw - f0) / h, (fs - f0) / h])
        step = np.linalg.solve(jac, -f0)
        w, sep = w + step[0], sep + step[1]
        if abs(step[0]) < tol * abs(w) and abs(step[1]) < tol * max(1.0, abs(sep)):
            return w, sep
    raise RuntimeError("Leaver iteration did not converge at a = %g" % (2 * a))


SCHWARZSCHILD = (2.0 * (0.3736716844 - 0.0889623157j), 4.0 + 0.0j)      # (omega, A) at a = 0 in 2M = 1 units (starting guess)


def kerr_qnm_220(spin, start=None):
    """M omega of the (2,2,0) mode at dimensionless spin a/M = `spin` in (-1, 1).  `start` = (spin0, M omega0, A0) continues
    from a known solution; without it the spin is walked up (or down) from Schwarzschild in steps of at most 0.05."""
    spin = float(spin)
    if not -1.0 < spin < 1.0:
        raise ValueError("spin must lie in (-1, 1)")
    if start is None:
        s0, w, sep = 0.0, SCHWARZSCHILD[0], SCHWARZSCHILD[1]
    else:
        s0, w, sep = start[0], 2.0 * start[1], start[2]
    steps = max(1, int(np.ceil(abs(spin - s0) / 0.05)))
    if abs(spin) > 0.9:
        steps = max(steps, int(np.ceil(abs(spin - s0) / 0.01)))
    for x in np.linspace(s0, spin, steps + 1)[1:] if spin != s0 else [spin]:
        w, sep = _newton(0.5 * x, w, sep)
    return 0.5 * w, sep


# ----------------------------------------------------------------------------------------
# the tabulated mode (what oracle.waveform reads)
# ----------------------------------------------------------------------------------------
TABLE_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "qnm_220_table.txt")
_cache = {}


def ringdown_table():
    """(spins, Re M omega, -Im M omega) from oracle/qnm_220_table.txt."""
    if "tab" not in _cache:
        data = np.loadtxt(TABLE_PATH)
        _cache["tab"] = (data[:, 0], data[:, 1], data[:, 2])
    return _cache["tab"]


def qnm_220(spin):
    """(Re M omega, -Im M omega) at `spin` by cubic-spline interpolation of the table (spin clamped to the table's range)."""
    from scipy.interpolate import CubicSpline
    if "spl" not in _cache:
        s, wr, wi = ringdown_table()
        _cache["spl"] = (CubicSpline(s, wr), CubicSpline(s, wi), s[0], s[-1])
    fr, fi, lo, hi = _cache["spl"]
    x = min(max(float(spin), lo), hi)
    return float(fr(x)), float(fi(x))
