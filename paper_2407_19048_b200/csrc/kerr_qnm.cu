// kerr_qnm.cu -- the l = m = 2, n = 0 quasi-normal mode of a Kerr black hole on a grid of spins (host code, run once
// per process when the first plan is created).
//
// IMRPhenomD (ref. [32]) places its ringdown at M f_RD = Re(omega)/2 pi, M f_damp = -Im(omega)/2 pi of
// this mode at the remnant's spin and interpolates tabulated values of it.  The library computes the tabulation itself:
// Leaver's continued-fraction conditions (Proc. R. Soc. A 402, 285 (1985); spin weight -2, units 2M = 1 inside the
// recurrences) for the angular and the radial Teukolsky equation are solved for (omega, A_lm) by Newton iteration, node
// after node, outwards from the Schwarzschild value.  Nodes are uniform in y = sqrt(1 - a/M) (the mode varies fastest
// towards the extremal hole): AMPLFI_QNM_NODES of them from a/M = +0.998 (y smallest) to -0.998; prepare_sample()
// interpolates with a four-point Lagrange cubic in y (relative error < 1e-7).
#include <cmath>
#include <complex>
#include <mutex>

#include "amplfi_internal.h"

namespace amplfi {

namespace {

using cd = std::complex<double>;
constexpr double kS = -2.0, kM = 2.0;

// value of beta_0 - alpha_0 gamma_1 / (beta_1 - alpha_1 gamma_2 / ...) for both recurrences
void leaver_conditions(cd w, cd sep, double a, int depth_radial, cd& f_ang, cd& f_rad) {
    const cd I(0.0, 1.0);
    const double b = std::sqrt(1.0 - 4.0 * a * a);
    const double k1 = 0.5 * std::fabs(kM - kS), k2 = 0.5 * std::fabs(kM + kS);
    {
        cd t = 0.0;
        for (int n = 120; n >= 0; --n) {
            const double dn = (double)n;
            const cd be = dn * (dn - 1.0) + 2.0 * dn * (k1 + k2 + 1.0 - 2.0 * a * w)
                          - (2.0 * a * w * (2.0 * k1 + kS + 1.0) - (k1 + k2) * (k1 + k2 + 1.0))
                          - (a * a * w * w + kS * (kS + 1.0) + sep);
            if (n == 0) { f_ang = be - t; break; }
            const double al_prev = -2.0 * dn * (dn - 1.0 + 2.0 * k1 + 1.0);          // alpha_{n-1}
            const cd ga = 2.0 * a * w * (dn + k1 + k2 + kS);
            t = al_prev * ga / (be - t);
        }
    }
    const cd q = 0.5 * w - a * kM;
    const cd c0 = 1.0 - kS - I * w - (2.0 * I / b) * q;
    const cd c1 = -4.0 + 2.0 * I * w * (2.0 + b) + (4.0 * I / b) * q;
    const cd c2 = kS + 3.0 - 3.0 * I * w - (2.0 * I / b) * q;
    const cd c3 = w * w * (4.0 + 2.0 * b - a * a) - 2.0 * a * kM * w - kS - 1.0 + (2.0 + b) * I * w - sep
                  + ((4.0 * w + 2.0 * I) / b) * q;
    const cd c4 = kS + 1.0 - 2.0 * w * w - (2.0 * kS + 3.0) * I * w - ((4.0 * w + 2.0 * I) / b) * q;
    cd t = 0.0;
    for (int n = depth_radial; n >= 0; --n) {
        const double dn = (double)n;
        const cd be = -2.0 * dn * dn + (c1 + 2.0) * dn + c3;
        if (n == 0) { f_rad = be - t; break; }
        const double dp = dn - 1.0;
        const cd al_prev = dp * dp + (c0 + 1.0) * dp + c0;
        const cd ga = dn * dn + (c2 - 3.0) * dn + c4 - c2 + 2.0;
        t = al_prev * ga / (be - t);
    }
}

bool newton(double a, cd& w, cd& sep) {
    const int depth = 400 + (int)(2600.0 * std::fmin(1.0, std::fmax(0.0, (std::fabs(2.0 * a) - 0.7) / 0.25)));
    for (int it = 0; it < 50; ++it) {
        cd fa0, fr0, fa1, fr1, fa2, fr2;
        const double h = 1e-7;
        leaver_conditions(w, sep, a, depth, fa0, fr0);
        leaver_conditions(w + h, sep, a, depth, fa1, fr1);
        leaver_conditions(w, sep + h, a, depth, fa2, fr2);
        const cd j00 = (fa1 - fa0) / h, j01 = (fa2 - fa0) / h, j10 = (fr1 - fr0) / h, j11 = (fr2 - fr0) / h;
        const cd det = j00 * j11 - j01 * j10;
        const cd dw = (-fa0 * j11 + fr0 * j01) / det, ds = (-fr0 * j00 + fa0 * j10) / det;
        w += dw;
        sep += ds;
        if (std::abs(dw) < 1e-13 * std::abs(w) && std::abs(ds) < 1e-13 * std::fmax(1.0, std::abs(sep))) return true;
    }
    return false;
}

double g_table[2 * AMPLFI_QNM_NODES];
bool g_ok = false;
std::once_flag g_once;

void build_table() {
    const double y_lo = std::sqrt(1.0 - 0.998), y_hi = std::sqrt(1.0 + 0.998);
    const double h = (y_hi - y_lo) / (AMPLFI_QNM_NODES - 1);
    // node nearest to a = 0 (y = 1), then outwards in both directions, each solve starting from its neighbour
    const int i0 = (int)std::lround((1.0 - y_lo) / h);
    bool ok = true;
    for (int dir = -1; dir <= 1; dir += 2) {
        cd w(2.0 * 0.3736716844, -2.0 * 0.0889623157), sep(4.0, 0.0);          // Schwarzschild, 2M = 1 units
        for (int i = (dir < 0 ? i0 : i0 + 1); i >= 0 && i < AMPLFI_QNM_NODES; i += dir) {
            const double y = y_lo + h * i, spin = 1.0 - y * y;
            if (!newton(0.5 * spin, w, sep)) ok = false;
            g_table[2 * i] = 0.5 * w.real();                                    // M omega
            g_table[2 * i + 1] = -0.5 * w.imag();
        }
    }
    g_ok = ok;
}

}  // namespace

// [AMPLFI_QNM_NODES][2] = (Re M omega, -Im M omega), node i at y = y_lo + i (y_hi - y_lo)/(NODES - 1); nullptr on failure
const double* kerr_qnm_table() {
    std::call_once(g_once, build_table);
    return g_ok ? g_table : nullptr;
}

}  // namespace amplfi
