// waveform.cuh -- per-sample waveform coefficients and the per-bin evaluator (device code).
//
// PAPER.md:87 (IMRPhenomD [32], inspiral = TaylorF2 3.5PN [33]) and PAPER.md:104 (waveforms are generated
// on the GPU).  The evaluation is split in two so that the hot loop is a handful of FMAs per bin:
//   1. prepare_sample(): one thread per sample, fp64.  Turns the 11 physical parameters into
//      coefficients of fixed powers of the BIN INDEX k (f_k = k/T): on a regular grid
//      (pi M f)^(p/3) = const * k^(p/3), so every PN / phenomenological term is
//      (per-sample constant) x (per-bin table value).
//   2. eval_h0(): per bin, phase in fp64 "turns" from k^(-1/3) and ln k (plan tables), reduced
//      modulo 1, then one fast sincos; amplitude in fp32.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace amplfi {

struct WfCoef {
    int valid, approx, k_lo, k_hi;           // k_lo > k_hi: empty band
    double kp1, kp2;                         // phase region boundaries in bins
    // region 1 (inspiral) phase / 2pi
    double lin1, c01, a_m5, a_m3, a_m2, a_m1, a_ln, a_p1, a_p1ln, a_p2, s_p4, s_p5, s_p6;
    // region 2 (intermediate)
    double lin2, c02, b_ln, b_m9;
    // region 3 (merger-ringdown)
    double lin3, c03, r_m3, r_34;
    float r_at, at_k0, at_invw;
    // amplitude
    float amp_scale, ka1, ka2;
    float e[8];                              // inspiral bracket: 1 + sum_{i=2..9} e[i-2] (k^(1/3))^i
    float q[5], q_mid, q_invh;               // intermediate quartic in u = (k - q_mid) * q_invh
    float g0, g_krd, g_invw, g2;             // ringdown: g0 exp(-g2 y)/(1 + y^2), y = (k - g_krd) g_invw
    float pol_p, pol_c;                      // (1 + cos^2 iota)/2, cos iota
};

struct DetResp { double fp, fc, dt; };

struct DetGeom { double r[3], x[3], y[3]; };

// Site constants (Earth-fixed, metres / unit vectors) for H1, L1, V1 (PAPER.md:13, :103 name the sites).
__device__ __constant__ DetGeom kDet[3] = {
    {{-2.16141492636e6, -3.83469517889e6, 4.60035022664e6},
     {-0.22389266154, 0.79983062746, 0.55690487831},
     {-0.91397818574, 0.02609403989, -0.40492342125}},
    {{-7.42760447238e4, -5.49628371971e6, 3.22425701744e6},
     {-0.95457412153, -0.14158077340, -0.26218911324},
     {0.29774156894, -0.48791033647, -0.82054461286}},
    {{4.54637409900e6, 8.42989697626e5, 4.37857696241e6},
     {-0.70045821479, 0.20848948619, 0.68256166277},
     {-0.05379255368, -0.96908180549, 0.24080451708}}};

#define AMPLFI_C_SI 299792458.0
#define AMPLFI_MTSUN 4.925490947641267e-06
#define AMPLFI_MPC 3.085677581491367e22
#define AMPLFI_GAMMA_E 0.5772156649015329
#define AMPLFI_PI 3.141592653589793238

// prepare_kernel runs one warp per SM through ~7000 straight-line instructions, so it is bound by instruction fetch
// (ncu: 45 % of its stall samples are "no instruction").  The fp64 library routines and the division are therefore kept
// out of line: one copy each, hit in the instruction cache from the second call on.
static __device__ __noinline__ double pexp(double x) { return exp(x); }
static __device__ __noinline__ double plog(double x) { return log(x); }
static __device__ __noinline__ double psqrt(double x) { return sqrt(x); }
static __device__ __noinline__ double pcos(double x) { return cos(x); }
static __device__ __noinline__ void psincos(double x, double* s, double* c) { sincos(x, s, c); }

// antenna patterns and geocentric delay of detector `det`
struct SkyFrame { double X[3], Y[3], n[3]; };

// polarisation axes X, Y and direction n toward the source in the Earth-fixed frame (shared by all detectors)
__device__ inline SkyFrame sky_frame(double ra, double dec, double psi, double gmst) {
    double sg, cg, sd, cd, sp, cp;
    psincos(gmst - ra, &sg, &cg);
    psincos(dec, &sd, &cd);
    psincos(psi, &sp, &cp);
    SkyFrame f;
    f.X[0] = -cp * sg - sp * cg * sd; f.X[1] = -cp * cg + sp * sg * sd; f.X[2] = sp * cd;
    f.Y[0] = sp * sg - cp * cg * sd;  f.Y[1] = sp * cg + cp * sg * sd;  f.Y[2] = cp * cd;
    f.n[0] = cd * cg; f.n[1] = -cd * sg; f.n[2] = sd;
    return f;
}

__device__ inline DetResp detector_response(const SkyFrame& f, int det) {
    const DetGeom& g = kDet[det];
    const double* X = f.X;
    const double* Y = f.Y;
    const double* n = f.n;
    // D = (x x^T - y y^T)/2 contracted with X, Y via the projections on the arms
    const double xX = g.x[0] * X[0] + g.x[1] * X[1] + g.x[2] * X[2];
    const double xY = g.x[0] * Y[0] + g.x[1] * Y[1] + g.x[2] * Y[2];
    const double yX = g.y[0] * X[0] + g.y[1] * X[1] + g.y[2] * X[2];
    const double yY = g.y[0] * Y[0] + g.y[1] * Y[1] + g.y[2] * Y[2];
    DetResp r;
    r.fp = 0.5 * ((xX * xX - yX * yX) - (xY * xY - yY * yY));
    r.fc = xX * xY - yX * yY;
    r.dt = -(g.r[0] * n[0] + g.r[1] * n[1] + g.r[2] * n[2]) / AMPLFI_C_SI;
    return r;
}

__device__ inline double pd_fit(const double* t, double eta, double xi) {
    const double e2 = eta * eta;
    return t[0] + t[1] * eta + xi * ((t[2] + t[3] * eta + t[4] * e2)
           + xi * ((t[5] + t[6] * eta + t[7] * e2) + xi * (t[8] + t[9] * eta + t[10] * e2)));
}

// p: 11 parameters; t_seg = n/fs; amp_mul multiplies the strain amplitude (1 for the API in strain/Hz).
// tab: [19][11] fit table in global/constant memory.
// Sine-Gaussian burst (reading R-W12): row = f0, Q, -, -, A, iota, phi, t0, ra, dec, psi.
//   h0(f_k) = A tau sqrt(pi)/2 exp(-(pi tau (f_k - f0))^2) exp(-i (2 pi f_k t0 - phi)),  tau = Q / (sqrt2 pi f0)
// Fields used: lin1 (t0/T, turns per bin), c01 (-phi / 2 pi), amp_scale, g_krd (f0 T), g_invw (pi tau / T), pol_p, pol_c.
__device__ inline void prepare_sine_gaussian(const double* p, double t_seg, int n_bins, double f_lo, double f_hi,
                                             double amp_mul, WfCoef& c) {
    const double PI = AMPLFI_PI;
    const double f0 = p[0], q = p[1], amp = p[4];
    bool ok = (f0 > 0.0) && (q > 0.0) && (amp > 0.0);
    for (int i = 0; i < 11; ++i) ok = ok && isfinite(p[i]);
    c.valid = ok ? 1 : 0;
    c.approx = 2;
    c.k_lo = 1;
    c.k_hi = 0;
    if (!ok) return;
    const double tau = q / (1.4142135623730951 * PI * f0);
    const double cosi = cos(p[5]);
    c.pol_p = (float)(0.5 * (1.0 + cosi * cosi));
    c.pol_c = (float)cosi;
    long klo = (long)ceil(f_lo * t_seg);
    while ((double)(klo - 1) / t_seg >= f_lo) --klo;
    while ((double)klo / t_seg < f_lo) ++klo;
    long khi = (long)floor(f_hi * t_seg);
    while ((double)(khi + 1) / t_seg <= f_hi) ++khi;
    while (khi >= 0 && (double)khi / t_seg > f_hi) --khi;
    if (klo < 1) klo = 1;
    if (khi > n_bins - 2) khi = n_bins - 2;
    c.k_lo = (int)klo;
    c.k_hi = (int)khi;
    c.lin1 = p[7] / t_seg;
    c.c01 = -p[6] / (2.0 * PI);
    c.amp_scale = (float)(amp_mul * 0.5 * amp * tau * 1.7724538509055159);      // sqrt(pi)
    c.g_krd = (float)(f0 * t_seg);
    c.g_invw = (float)(PI * tau / t_seg);
}

__device__ __forceinline__ float2 eval_sine_gaussian(const WfCoef& c, int k) {
    double ph = fma(c.lin1, (double)k, c.c01);
    ph -= rint(ph);
    float s, co;
    __sincosf((float)ph * 6.283185307179586f, &s, &co);
    const float y = ((float)k - c.g_krd) * c.g_invw;
    const float amp = c.amp_scale * __expf(-y * y);
    return make_float2(amp * co, -amp * s);
}

// ROLE: bit 0 = the phase fields of WfCoef (and validity, band, polarisation factors), bit 1 = the amplitude fields.
// prepare_kernel runs the two halves in different warps (each recomputes the few quantities both need), which halves the
// dependent fp64 chain a sample waits for; whatever feeds only the other role's fields is removed by the compiler, the
// out-of-line library calls are guarded explicitly.
#define WF_PHASE 1
#define WF_AMP 2
template <int ROLE>
__device__ __forceinline__ void prepare_sample(const double* p, int approx, double t_seg, int n_bins, double f_lo,
                                               double f_hi, double amp_mul, const double* tab, WfCoef& c) {
    if (approx == 2) { prepare_sine_gaussian(p, t_seg, n_bins, f_lo, f_hi, amp_mul, c); return; }
    const double PI = AMPLFI_PI, TWO_PI = 2.0 * AMPLFI_PI, I2PI = 0.15915494309189535;   // 1 / (2 pi)
    const double mc = p[0], q = p[1], chi1 = p[2], chi2 = p[3], dist = p[4];
    bool ok = (mc > 0.0) && (q > 0.0) && (q <= 1.0) && (fabs(chi1) < 1.0) && (fabs(chi2) < 1.0) && (dist > 0.0);
    for (int i = 0; i < 11; ++i) ok = ok && isfinite(p[i]);
    c.valid = ok ? 1 : 0;
    c.approx = approx;
    c.k_lo = 1;
    c.k_hi = 0;
    if (!ok) return;
    const double eta = q / ((1.0 + q) * (1.0 + q));
    const double ieta = 1.0 / eta;                   // reciprocals once: every fp64 division is ~25 instructions of this
                                                     // fetch-bound kernel
    const double mtot = mc * pexp(-0.6 * plog(eta));
    const double ms = mtot * AMPLFI_MTSUN;           // seconds
    const double mu = ms / t_seg;                    // Mf = mu * k
    const double imu = 1.0 / mu;
    const double lnmu = plog(mu);
    const double lnv1 = (lnmu + 1.1447298858494002) * (1.0 / 3.0);     // ln(pi) = 1.14472988584940017...
    const double v1 = pexp(lnv1);                     // (pi mu)^(1/3): v = v1 * k^(1/3)
    const double cosi = pcos(p[5]);
    c.pol_p = (float)(0.5 * (1.0 + cosi * cosi));
    c.pol_c = (float)cosi;

    // ---- band (DESIGN.md R-W7): f_lo <= k/T <= f_top, 1 <= k <= n_bins-2 ----
    const double f_top = fmin(approx == 0 ? 1.0 / (14.696938456699069 * PI * ms) : 0.2 / ms, f_hi);   // 6^(3/2)
    long klo = (long)ceil(f_lo * t_seg);
    while ((double)(klo - 1) / t_seg >= f_lo) --klo;
    while ((double)klo / t_seg < f_lo) ++klo;
    long khi = (long)floor(f_top * t_seg);
    while ((double)(khi + 1) / t_seg <= f_top) ++khi;
    while (khi >= 0 && (double)khi / t_seg > f_top) --khi;
    if (klo < 1) klo = 1;
    if (khi > n_bins - 2) khi = n_bins - 2;
    c.k_lo = (int)klo;
    c.k_hi = (int)khi;

    // ---- TaylorF2 phasing series (aligned spins for IMRPhenomD, none for TaylorF2) ----
    const double s1 = (approx == 0) ? 0.0 : chi1, s2 = (approx == 0) ? 0.0 : chi2;
    const double seta = psqrt(fmax(1.0 - 4.0 * eta, 0.0));
    const double m1 = 0.5 * (1.0 + seta), m2 = 0.5 * (1.0 - seta);
    const double SL = m1 * m1 * s1 + m2 * m2 * s2;
    const double dSL = (m1 - m2) * (m2 * s2 - m1 * s1);
    const double e2 = eta * eta, e3 = e2 * eta;
    // (divisions by constants are written as multiplications by the reciprocal: an fp64 division is ~25 dependent instructions)
    double pv2 = (5.0 / 9.0) * (743.0 / 84.0 + 11.0 * eta);
    double pv3 = -16.0 * PI + (188.0 / 3.0) * SL + 25.0 * dSL;
    const double sig = eta * (721.0 / 48.0 - 247.0 / 48.0) * s1 * s2
                       + (719.0 / 96.0 - 233.0 / 96.0) * (m1 * m1 * s1 * s1 + m2 * m2 * s2 * s2);
    double pv4 = (5.0 / 72.0) * (3058.673 / 7.056 + 5429.0 / 7.0 * eta + 617.0 * e2) - 10.0 * sig;
    const double gam = (554345.0 / 1134.0 + (110.0 / 9.0) * eta) * SL + (13915.0 / 84.0 - (10.0 / 3.0) * eta) * dSL;
    double pv5 = 5.0 / 9.0 * (7729.0 / 84.0 - 13.0 * eta) * PI - gam;
    double pl5 = 5.0 / 3.0 * (7729.0 / 84.0 - 13.0 * eta) * PI - 3.0 * gam;
    double pv6 = 11583.231236531 / 4.694215680 - 640.0 / 3.0 * PI * PI - 6848.0 / 21.0 * AMPLFI_GAMMA_E
                 + eta * (-15737.765635 / 3.048192 + 2255.0 / 12.0 * PI * PI) + e2 * (76055.0 / 1728.0)
                 - e3 * (127825.0 / 1296.0) - 6848.0 / 21.0 * 1.3862943611198906        /* ln 4 */
                 + (PI / 3.0) * (3760.0 * SL + 1490.0 * dSL);
    double pl6 = -6848.0 / 21.0;
    double pv7 = PI * (77096675.0 / 254016.0 + 378515.0 / 1512.0 * eta - 74045.0 / 756.0 * e2)
                 + (-8980424995.0 / 762048.0 + (6586595.0 / 756.0) * eta - (305.0 / 36.0) * e2) * SL
                 - (170978035.0 / 48384.0 - (2876425.0 / 672.0) * eta - (4735.0 / 144.0) * e2) * dSL;
    const double pfa = 3.0 / 128.0 * ieta * I2PI;          // everything below is in turns
    const double iv = 1.0 / v1;
    c.a_m5 = pfa * iv * iv * iv * iv * iv;
    c.a_m3 = pfa * pv2 * iv * iv * iv;
    c.a_m2 = pfa * pv3 * iv * iv;
    c.a_m1 = pfa * pv4 * iv;
    c.a_ln = pfa * pl5 * (1.0 / 3.0);
    c.a_p1 = pfa * (pv6 + pl6 * lnv1) * v1;
    c.a_p1ln = pfa * pl6 * (1.0 / 3.0) * v1;
    c.a_p2 = pfa * pv7 * v1 * v1;
    const double tc_turns = p[7] / t_seg;                     // 2 pi f t_c / 2 pi = k t_c / T
    const double phic_turns = -2.0 * p[6] * I2PI;
    double const1 = pfa * (pv5 + pl5 * lnv1) - 0.125 + phic_turns;      // -pi/4 -> -1/8 turn

    if (approx == 0) {
        c.kp1 = 1e300; c.kp2 = 1e300;
        c.lin1 = tc_turns; c.c01 = const1;
        c.s_p4 = c.s_p5 = c.s_p6 = 0.0;
        c.lin2 = c.c02 = c.b_ln = c.b_m9 = 0.0;
        c.lin3 = c.c03 = c.r_m3 = c.r_34 = 0.0;
        c.r_at = 0.f; c.at_k0 = 0.f; c.at_invw = 0.f;
        // A0 f^(-7/6), A0 = sqrt(5/24) pi^(-2/3) (G Mc/c^3)^(5/6) c / D
        if (ROLE & WF_AMP) {
            const double a0 = 0.45643546458763845 /* sqrt(5/24) */ * 0.46619407703541166 /* pi^(-2/3) */ * pow(mc * AMPLFI_MTSUN, 5.0 / 6.0)
                              * AMPLFI_C_SI / (dist * AMPLFI_MPC);
            c.amp_scale = (float)(a0 * pow(t_seg, 7.0 / 6.0) * amp_mul);
        }
        c.ka1 = 3.0e38f; c.ka2 = 3.0e38f;
        for (int i = 0; i < 8; ++i) c.e[i] = 0.f;
        for (int i = 0; i < 5; ++i) c.q[i] = 0.f;
        c.q_mid = 0.f; c.q_invh = 0.f; c.g0 = 0.f; c.g_krd = 0.f; c.g_invw = 0.f; c.g2 = 0.f;
        return;
    }

    // ---- IMRPhenomD ----
    const double xi = (m1 * chi1 + m2 * chi2 - (38.0 / 113.0) * eta * (chi1 + chi2)) - 1.0;
    double fit[AMPLFI_PD_ROWS];
#pragma unroll
    for (int r = 0; r < AMPLFI_PD_ROWS; ++r) fit[r] = pd_fit(tab + r * AMPLFI_PD_COLS, eta, xi);
    // remnant: final spin, radiated energy, ringdown / damping frequency (Kerr 220 closed-form fit)
    const double stot = m1 * m1 * chi1 + m2 * m2 * chi2;
    const double e4 = e2 * e2;
    double af = 3.4641016151377544 * eta - 4.399247300629289 * e2 + 9.397292189321194 * e3 - 13.180949901606242 * e4
                + (1.0 - 0.0850917821418767 * eta - 5.837029316602263 * e2) * stot
                + (0.1014665242971878 * eta - 2.0967746996832157 * e2) * stot * stot
                + (-1.3546806617824356 * eta + 4.108962025369336 * e2) * stot * stot * stot
                + (-0.8676969352555539 * eta + 2.064046835273906 * e2) * stot * stot * stot * stot;
    af = fmin(fmax(af, -0.998), 0.998);                    // the mode table's range
    const double sn = stot / (m1 * m1 + m2 * m2);
    const double erad = (eta * (0.055974469826360077 + 0.5809510763115132 * eta - 0.9606726679372312 * e2
                                + 3.352411249771192 * e3)
                         * (1.0 + (-0.0030302335878845507 - 2.0066110851351073 * eta + 7.7050567802399215 * e2) * sn))
                        / (1.0 + (-0.6714403054720589 - 1.4756929437702908 * eta + 7.304676214885011 * e2) * sn);
    // Kerr (2,2,0) mode at the final spin: four-point Lagrange cubic on the plan's table (kerr_qnm.cu; nodes uniform in
    // y = sqrt(1 - a), from a = +0.998 down to -0.998), f_RD = Re(omega)/2 pi, f_damp = -Im(omega)/2 pi per remnant mass
    double w_re, w_im;
    {
        const double* qnm = tab + AMPLFI_QNM_OFFSET;
        const double y_lo = 0.044721359549995794 /* sqrt(0.002) */, y_hi = 1.4135062787267694 /* sqrt(1.998) */;
        const double inv_h = (double)(AMPLFI_QNM_NODES - 1) / (y_hi - y_lo);
        const double u = (psqrt(1.0 - af) - y_lo) * inv_h;
        int i = (int)floor(u);
        i = i < 1 ? 1 : (i > AMPLFI_QNM_NODES - 3 ? AMPLFI_QNM_NODES - 3 : i);
        const double t = u - (double)i;
        const double l0 = -t * (t - 1.0) * (t - 2.0) * (1.0 / 6.0), l1 = (t + 1.0) * (t - 1.0) * (t - 2.0) * 0.5;
        const double l2 = -(t + 1.0) * t * (t - 2.0) * 0.5, l3 = (t + 1.0) * t * (t - 1.0) * (1.0 / 6.0);
        const double* q = qnm + 2 * (i - 1);
        w_re = l0 * q[0] + l1 * q[2] + l2 * q[4] + l3 * q[6];
        w_im = l0 * q[1] + l1 * q[3] + l2 * q[5] + l3 * q[7];
    }
    const double imf = 1.0 / (1.0 - erad);           // remnant mass
    const double f_rd = w_re * I2PI * imf;
    const double f_dm = w_im * I2PI * imf;
    // amplitude peak (both roles: the phase is aligned in time there)
    const double g1 = fit[PD_GAMMA1], g2 = fit[PD_GAMMA2], g3 = fit[PD_GAMMA3];
    const double f_peak = (g2 > 1.0) ? fabs(f_rd - f_dm * g3 / g2)
                                     : fabs(f_rd + f_dm * (psqrt(1.0 - g2 * g2) - 1.0) * g3 / g2);
    const double mu13 = v1 * 0.6827840632552957;      // mu^(1/3) = (pi mu)^(1/3) pi^(-1/3)

    if (ROLE & WF_PHASE) {

    const double sg1 = fit[PD_SIGMA1], sg2 = fit[PD_SIGMA2], sg3 = fit[PD_SIGMA3], sg4 = fit[PD_SIGMA4];
    const double be1 = fit[PD_BETA1], be2 = fit[PD_BETA2], be3 = fit[PD_BETA3];
    const double al1 = fit[PD_ALPHA1], al2 = fit[PD_ALPHA2], al3 = fit[PD_ALPHA3], al4 = fit[PD_ALPHA4],
                 al5 = fit[PD_ALPHA5];
    // phases in radians as functions of Mf (value, derivative) at the two junctions
    const double pn[8] = {1.0, 0.0, pv2, pv3, pv4, pv5, pv6, pv7};
    const double pl[8] = {0.0, 0.0, 0.0, 0.0, 0.0, pl5, pl6, 0.0};
    const double pfar = 3.0 / 128.0 * ieta;
    const double f1 = 0.018, f2 = 0.5 * f_rd;
    double phi_ins, dphi_ins;
    {
        // the junction frequencies are constants of the model: their roots and logarithms are written out
        const double v = 0.3838316585355026 /* cbrt(pi 0.018) */, lv = -0.957551211745524 /* ln v */;
        double s = 0.0, ds = 0.0, vp = 1.0 / (v * v * v * v * v * v);      // v^(i-6)
        for (int i = 0; i < 8; ++i) {
            s += (pn[i] + pl[i] * lv) * vp * v;                            // v^(i-5)
            ds += ((i - 5) * (pn[i] + pl[i] * lv) + pl[i]) * vp;
            vp *= v;
        }
        const double c13 = 0.26207413942088964;   // cbrt(0.018)
        phi_ins = pfar * s - PI / 4.0
                  + (sg1 * f1 + 0.75 * sg2 * f1 * c13 + 0.6 * sg3 * f1 * c13 * c13 + 0.5 * sg4 * f1 * f1) * ieta;
        dphi_ins = pfar * ds * (v / (3.0 * f1)) + (sg1 + sg2 * c13 + sg3 * c13 * c13 + sg4 * f1) * ieta;
    }
    const double if1 = 1.0 / 0.018, if1_3 = if1 * if1 * if1;      // constant: folded at compile time
    const double int1 = (be1 * f1 + be2 * -4.017383521085972 /* ln 0.018 */ - be3 * if1_3 * (1.0 / 3.0)) * ieta;
    const double dint1 = (be1 + be2 * if1 + be3 * if1_3 * if1) * ieta;
    const double c2int = dphi_ins - dint1;
    const double c1int = phi_ins - int1 - c2int * f1;
    const double lnf2 = plog(f2), f2m14 = rsqrt(psqrt(f2));                   // f2^(-1/4)
    const double if2 = 1.0 / f2, if2_3 = if2 * if2 * if2;
    const double int2 = (be1 * f2 + be2 * lnf2 - be3 * if2_3 * (1.0 / 3.0)) * ieta + c1int + c2int * f2;
    const double dint2 = (be1 + be2 * if2 + be3 * if2_3 * if2) * ieta + c2int;
    const double ifdm = 1.0 / f_dm;
    const double x2 = (f2 - al5 * f_rd) * ifdm;
    const double mr2 = (al1 * f2 - al2 * if2 + 4.0 / 3.0 * al3 * (f2 * f2m14) + al4 * atan(x2)) * ieta;
    const double dmr2 = (al1 + al2 * if2 * if2 + al3 * f2m14 + al4 * ifdm / (1.0 + x2 * x2)) * ieta;
    const double c2mr = dint2 - dmr2;
    const double c1mr = int2 - mr2 - c2mr * f2;
    // time alignment at the amplitude peak
    const double xp = (f_peak - al5 * f_rd) * ifdm;
    const double t0 = (al1 + al2 / (f_peak * f_peak) + al3 * rsqrt(psqrt(f_peak)) + al4 * ifdm / (1.0 + xp * xp)) * ieta
                      + c2mr;

    c.kp1 = f1 * imu;
    c.kp2 = f2 * imu;
    c.lin1 = tc_turns + (sg1 * ieta - t0) * mu * I2PI;
    c.c01 = const1;
    c.s_p4 = 0.75 * sg2 * ieta * mu * mu13 * I2PI;
    c.s_p5 = 0.6 * sg3 * ieta * mu * mu13 * mu13 * I2PI;
    c.s_p6 = 0.5 * sg4 * ieta * mu * mu * I2PI;
    c.lin2 = tc_turns + (be1 * ieta + c2int - t0) * mu * I2PI;
    c.c02 = (c1int + be2 * ieta * lnmu) * I2PI + phic_turns;
    c.b_ln = be2 * ieta * I2PI;
    c.b_m9 = -be3 * (1.0 / 3.0) * ieta * imu * imu * imu * I2PI;
    c.lin3 = tc_turns + (al1 * ieta + c2mr - t0) * mu * I2PI;
    c.c03 = c1mr * I2PI + phic_turns;
    c.r_m3 = -al2 * ieta * imu * I2PI;
    c.r_34 = 4.0 / 3.0 * al3 * ieta * pexp(0.75 * lnmu) * I2PI;
    c.r_at = (float)(al4 * ieta * I2PI);
    c.at_k0 = (float)(al5 * f_rd * imu);
    c.at_invw = (float)(mu * ifdm);
    }
    if (!(ROLE & WF_AMP)) return;

    // ---- amplitude ----
    const double amp0 = 2.0 * 0.15769578262626002 /* sqrt(5 / (64 pi)) */ * mtot * mtot * AMPLFI_MTSUN * (AMPLFI_MTSUN * AMPLFI_C_SI)
                        / (dist * AMPLFI_MPC);
    c.amp_scale = (float)(amp0 * psqrt(eta * (2.0 / 3.0)) * 0.8263074871107581 * pexp(-7.0 / 6.0 * lnmu) * amp_mul);   // pi^(-1/6)
    const double c12 = chi1 * chi1, c22 = chi2 * chi2;
    double A[7];
    A[2] = (-969.0 + 1804.0 * eta) * (1.0 / 672.0);
    A[3] = (chi1 * (81.0 * (1.0 + seta) - 44.0 * eta) + chi2 * (81.0 - 81.0 * seta - 44.0 * eta)) * (1.0 / 48.0);
    A[4] = (-27312085.0 - 10287648.0 * c22 - 10287648.0 * c12 * (1.0 + seta) + 10287648.0 * c22 * seta
            + 24.0 * (-1975055.0 + 857304.0 * c12 - 994896.0 * chi1 * chi2 + 857304.0 * c22) * eta
            + 35371056.0 * e2) * (1.0 / 8128512.0);
    A[5] = (chi2 * (-285197.0 * (-1.0 + seta) + 4.0 * (-91902.0 + 1579.0 * seta) * eta - 35632.0 * e2)
            + chi1 * (285197.0 * (1.0 + seta) - 4.0 * (91902.0 + 1579.0 * seta) * eta - 35632.0 * e2)
            + 42840.0 * (-1.0 + 4.0 * eta) * PI) * (1.0 / 32256.0);
    A[6] = -(-336.0 * (-3248849057.0 + 2943675504.0 * c12 - 3339284256.0 * chi1 * chi2 + 2943675504.0 * c22) * e2
             - 324322727232.0 * e3
             - 7.0 * (-177520268561.0 + 107414046432.0 * c22 + 107414046432.0 * c12 * (1.0 + seta)
                      - 107414046432.0 * c22 * seta + 11087290368.0 * (chi1 + chi2 + chi1 * seta - chi2 * seta) * PI)
             + 12.0 * eta * (-545384828789.0 - 176491177632.0 * chi1 * chi2 + 202603761360.0 * c22
                             + 77616.0 * c12 * (2610335.0 + 995766.0 * seta) - 77287373856.0 * c22 * seta
                             + 5841690624.0 * (chi1 + chi2) * PI + 21384760320.0 * PI * PI)) * (1.0 / 60085960704.0);
    const double rho1 = fit[PD_RHO1], rho2 = fit[PD_RHO2], rho3 = fit[PD_RHO3];
    {
        double vp = v1 * v1;
        for (int i = 2; i <= 6; ++i) { c.e[i - 2] = (float)(A[i] * vp); vp *= v1; }
        c.e[5] = (float)(rho1 * mu * mu * mu13);                // Mf^(7/3) = mu^(7/3) k^(7/3)
        c.e[6] = (float)(rho2 * mu * mu * mu13 * mu13);
        c.e[7] = (float)(rho3 * mu * mu * mu);
    }
    // inspiral bracket and slope at Mf = 0.014; ringdown ansatz value and slope at f_peak
    const double fa = 0.014, fc = f_peak;
    double va, da;
    {
        const double x = 0.35298748079802034 /* cbrt(pi 0.014) */, dx = x / (3.0 * fa), c13 = 0.24101422641752301 /* cbrt(0.014) */;
        va = 1.0 + x * x * (A[2] + x * (A[3] + x * (A[4] + x * (A[5] + x * A[6]))))
             + fa * fa * c13 * (rho1 + c13 * (rho2 + c13 * rho3));
        da = (2.0 * A[2] * x + 3.0 * A[3] * x * x + 4.0 * A[4] * x * x * x + 5.0 * A[5] * x * x * x * x
              + 6.0 * A[6] * x * x * x * x * x) * dx
             + 7.0 / 3.0 * rho1 * fa * c13 + 8.0 / 3.0 * rho2 * fa * c13 * c13 + 3.0 * rho3 * fa * fa;
    }
    const double w = f_dm * g3;
    double vc, dc;
    {
        const double d = fc - f_rd;
        const double iw = 1.0 / w, ilor = 1.0 / (d * d + w * w);
        const double lor = w * g1 * ilor;
        const double ex = pexp(-d * g2 * iw);
        vc = ex * lor;
        dc = ex * lor * (-g2 * iw - 2.0 * d * ilor);
    }
    // quartic through (fa: value, slope), (midpoint: v2), (fc: value, slope) in u = (f - fm)/h in [-1, 1]
    const double h = 0.5 * (fc - fa), fm = 0.5 * (fc + fa), vm = fit[PD_V2];
    const double S = 0.5 * (vc + va) - vm, Aodd = 0.5 * (vc - va);
    const double Dp = 0.5 * (dc + da) * h, Dm = 0.5 * (dc - da) * h;
    const double q3 = 0.5 * (Dp - Aodd), q1 = Aodd - q3, q4 = 0.5 * (Dm - 2.0 * S), q2 = S - q4;
    c.q[0] = (float)vm; c.q[1] = (float)q1; c.q[2] = (float)q2; c.q[3] = (float)q3; c.q[4] = (float)q4;
    c.q_mid = (float)(fm * imu);
    c.q_invh = (float)(mu / h);
    c.ka1 = (float)(fa * imu);
    c.ka2 = (float)(fc * imu);
    c.g0 = (float)(g1 / w);
    c.g_krd = (float)(f_rd * imu);
    c.g_invw = (float)(mu / w);
    c.g2 = (float)g2;
}

// MUFU approximations without the subnormal fix-ups of the library wrappers (every argument here is a normal number or
// may flush to zero): ~12 instructions per bin of an instruction-bound kernel
__device__ __forceinline__ float rsq_approx(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float exp_approx(float x) {
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x * 1.4426950408889634f));
    return r;
}

// h0 at bin k (k_lo <= k <= k_hi assumed).  ci = k^(-1/3), lnk = ln k (fp64 tables of the plan).
__device__ __forceinline__ float2 eval_h0(const WfCoef& c, int k, double ci, double lnk) {
    const double kd = (double)k;
    const double ci2 = ci * ci;
    const double c1 = kd * ci2;                       // k^(1/3)
    double ph;
    if (kd < c.kp1) {
        ph = fma(c.lin1, kd, c.c01);
        ph = fma(c.a_ln, lnk, ph);
        ph = fma(ci, fma(ci, fma(ci, fma(ci2, c.a_m5, c.a_m3), c.a_m2), c.a_m1), ph);
        ph = fma(c1, fma(c1, c.a_p2, fma(c.a_p1ln, lnk, c.a_p1)), ph);
        if (c.approx != 0) ph = fma(kd * c1, fma(c1, fma(c1, c.s_p6, c.s_p5), c.s_p4), ph);
    } else if (kd < c.kp2) {
        const double ci3 = ci2 * ci;
        ph = fma(c.lin2, kd, c.c02);
        ph = fma(c.b_ln, lnk, ph);
        ph = fma(c.b_m9, ci3 * ci3 * ci3, ph);
    } else {
        // k^(3/4) = k * k^(-1/4): fp32 seed (two MUFU) and one Newton step in fp64 (relative error ~1e-13),
        // instead of two software fp64 square roots
        const float kq = (float)k;
        const double y0 = (double)rsq_approx(kq * rsq_approx(kq));      // ~k^(-1/4), two MUFU, no slow paths
        const double y2 = y0 * y0;
        const double y1 = fma(0.25 * y0, fma(-kd, y2 * y2, 1.0), y0);
        ph = fma(c.lin3, kd, c.c03);
        ph = fma(c.r_m3, ci2 * ci, ph);
        ph = fma(c.r_34, kd * y1, ph);
        ph += (double)(c.r_at * atanf(((float)k - c.at_k0) * c.at_invw));
    }
    ph -= rint(ph);                                   // turns in [-1/2, 1/2]
    float s, co;
    __sincosf((float)ph * 6.283185307179586f, &s, &co);

    const float kf = (float)k, cf = (float)ci, c1f = (float)c1;
    const float cf2 = cf * cf;
    float amp = c.amp_scale * cf2 * cf2 * rsq_approx(cf);    // k^(-7/6) = cf^(7/2), cf = k^(-1/3)
    if (kf < c.ka1) {
        float br = c.e[7];
#pragma unroll
        for (int i = 6; i >= 0; --i) br = fmaf(br, c1f, c.e[i]);
        amp *= fmaf(br, c1f * c1f, 1.0f);
    } else if (kf < c.ka2) {
        const float u = (kf - c.q_mid) * c.q_invh;
        amp *= fmaf(u, fmaf(u, fmaf(u, fmaf(u, c.q[4], c.q[3]), c.q[2]), c.q[1]), c.q[0]);
    } else {
        const float y = (kf - c.g_krd) * c.g_invw;
        amp *= c.g0 * exp_approx(-c.g2 * y) * rcp_approx(fmaf(y, y, 1.0f));
    }
    return make_float2(amp * co, -amp * s);           // A exp(-i Psi)
}

}  // namespace amplfi
