/*
 * amplfi.h -- C ABI of libamplfi: the GPU data-generation hot path of AMPLFI
 * (arXiv 2407.19048, section 3 "Simulations on Accelerated Hardware").
 *
 * Every step of the path runs in hand-written CUDA kernels for sm_100a (B200).  There is no
 * CPU fallback: without a CUDA device every compute call returns AMPLFI_ERR_CUDA.
 *
 * Conventions ("Boundary"):
 *  - Every pointer argument below is a DEVICE pointer unless its comment says HOST.
 *  - All buffers are owned by the caller, row-major, contiguous.  Complex numbers are interleaved
 *    (re, im) float pairs.  The library allocates device memory only in amplfi_plan_create (tables,
 *    Welch partial sums, per-sample coefficient workspace) and frees it in amplfi_plan_destroy.
 *  - Calls enqueue work on the caller's stream (`stream` is a cudaStream_t passed as void*, NULL = the
 *    legacy default stream) and return without synchronising.  A plan must not be used from two
 *    streams at once (its workspace is shared).
 *  - Return value: AMPLFI_OK or a negative AMPLFI_ERR_*; amplfi_last_error() gives a thread-local
 *    message.  No exceptions, no aborts, nothing printed.
 *  - Units: masses in solar masses, distance in Mpc, times in seconds, angles in radians.
 *    Strain buffers (noise, bg, strip) are fp32 in natural strain units (~1e-21).  Frequency-domain
 *    waveform buffers (hp, hc, h_det) are fp32 in strain/Hz.  Power spectra do not fit fp32's range
 *    (S ~ 1e-47 strain^2/Hz): every `psd` buffer holds  S(f) * 2^140  (amplfi_psd_scale()).
 *    Whitened output is dimensionless (unit variance per kept frequency bin).
 *  - Frequency grid of a plan: f_k = k * fs / n, k = 0 .. K-1, K = n/2 + 1.
 *  - Fourier convention: forward X[k] = sum_n x[n] exp(-2 pi i k n / N); a signal
 *    h(f) = A exp(-i Psi), Psi containing +2 pi f t_c, merges at time t_c inside the segment.
 */
#ifndef AMPLFI_H
#define AMPLFI_H

#ifdef __cplusplus
extern "C" {
#endif

#define AMPLFI_OK                    0
#define AMPLFI_ERR_INVALID_ARG      (-1)  /* null pointer, batch/n_det <= 0, f_lo >= f_hi, f_hi > fs/2, bad ids */
#define AMPLFI_ERR_UNSUPPORTED_SIZE (-2)  /* n not a power of two in [2^10, 2^20], nperseg not one in [2^10, 2^15]; nperseg > n_bg */
#define AMPLFI_ERR_CUDA             (-3)  /* CUDA runtime/launch error (message in amplfi_last_error) */
#define AMPLFI_ERR_ALIGNMENT        (-4)  /* a buffer is not aligned as documented */

#define AMPLFI_TAYLORF2    0   /* 3.5PN non-spinning inspiral to f_ISCO (ref. [33]) */
#define AMPLFI_IMRPHENOMD  1   /* the paper's approximant (ref. [32]), aligned spins */
#define AMPLFI_SINE_GAUSSIAN 2 /* burst family the paper names as an extension; see the params note below */

#define AMPLFI_H1 0
#define AMPLFI_L1 1
#define AMPLFI_V1 2

#define AMPLFI_N_PARAMS 11
/* params row (fp64): 0 mchirp  1 q = m2/m1 in (0,1]  2 chi1  3 chi2  4 dist_mpc  5 theta_jn  6 phi_c
 *                    7 t_c (seconds from the start of the segment)  8 ra  9 dec  10 psi
 * = Theta of PAPER.md:151 eq. (4) plus the aligned spins and the arrival time
 * (PAPER.md:93, :117).  A row with q outside (0,1], |chi| >= 1, dist <= 0, mchirp <= 0 or a
 * non-finite entry does not fail the call: that sample's waveform is identically zero and
 * flags[b] = 1 where a flags buffer is given.
 * AMPLFI_SINE_GAUSSIAN reads the row as  0 f0 [Hz]  1 Q  2,3 unused  4 peak amplitude A  5 iota (ellipticity angle)
 * 6 phi  7 t0 (central time)  8 ra  9 dec  10 psi  and evaluates, with tau = Q / (sqrt2 pi f0),
 *     h0(f) = A tau sqrt(pi)/2 exp(-(pi tau (f - f0))^2) exp(-i (2 pi f t0 - phi)),  h+ = (1+cos^2 iota)/2 h0,  hx = -i cos iota h0,
 * the Fourier transform of  h+(t) = (1+cos^2 iota)/2 A e^{-(t-t0)^2/tau^2} cos(2 pi f0 (t-t0) + phi),
 * hx(t) = cos iota A e^{-(t-t0)^2/tau^2} sin(2 pi f0 (t-t0) + phi)  up to the mirror term at -f0 (<= e^{-Q^2/2} of the peak);
 * invalid: f0 <= 0, Q <= 0, A <= 0 or a non-finite entry. */

typedef struct amplfi_plan amplfi_plan;   /* opaque */

/* Thread-local description of the last error returned on this thread ("" if none). HOST string. */
const char* amplfi_last_error(void);

/* 2^140, the factor every psd buffer is multiplied by. */
double amplfi_psd_scale(void);

/* Library build tag, e.g. "amplfi-b200 sm_100a". HOST string. */
const char* amplfi_version(void);

/* Copy of the IMRPhenomD fit table the kernels use: 19 rows x 11 doubles, row order
 * rho1 rho2 rho3 v2 gamma1 gamma2 gamma3 sigma1..4 beta1..3 alpha1..5.  `out` is a HOST buffer of
 * 209 doubles.  (Used by the tests to check the library's copy against the oracle's.) */
int amplfi_phenomd_table(double* out);

/* The Kerr l = m = 2, n = 0 quasi-normal mode the IMRPhenomD ringdown uses (ref. [32]), as
 * the library tabulates it at first use (Leaver's continued fractions, csrc/kerr_qnm.cu): 512 nodes uniform in
 * y = sqrt(1 - a/M) from a/M = +0.998 (node 0) down to -0.998; `out` is a HOST buffer of 1024 doubles receiving
 * (Re M omega, -Im M omega) per node.  Returns the node count, or a negative status.  M f_RD = Re/(2 pi),
 * M f_damp = -Im/(2 pi) per remnant mass, interpolated with a four-point Lagrange cubic in y.
 * Conventions of the approximant (reading R-W1 of DESIGN.md): Psi(f) = 2 pi f t_c - 2 phi_c + phi_IMR(Mf) - t0 Mf with
 * t0 = d phi_IMR / d(Mf) at the amplitude peak f_peak INCLUDING the C1-junction constant of the merger-ringdown
 * region (the true phase derivative there), so that the time-domain amplitude peak sits at t_c; there is no
 * reference-frequency term. */
int amplfi_qnm_table(double* out);

/* Create a plan for segments of n samples at fs Hz seen by n_det detectors.
 *   n        power of two, 2^10 .. 2^20 (4 s at 2048 Hz = 8192; minutes-long
 *            binary-neutron-star segments are "larger by an order of magnitude": 256 s at 4096 Hz = 2^20)
 *   det_ids  HOST array [n_det] of AMPLFI_H1/L1/V1 ("Hanford and Livingston"), n_det 1..3
 *   max_batch  largest batch later passed to the per-batch calls (sizes the coefficient workspace
 *              and, for the fused call, the [max_batch, K] complex h0 workspace)
 *   nperseg  Welch segment length, power of two 2^10 .. 2^15 with nperseg <= n, or 0 if
 *            amplfi_psd_welch will not be called
 * Allocates device tables on the current CUDA device.  *out receives the plan. */
int amplfi_plan_create(int n, double fs, int n_det, const int* det_ids, int max_batch, int nperseg,
                       amplfi_plan** out);
void amplfi_plan_destroy(amplfi_plan* plan);

/* a-1 Waveform (section 3.1; "generate the IMRPhenomD waveforms directly on
 * the GPU").  For each sample b and bin k:
 *     h+ = (1 + cos^2 theta_jn)/2 * h0,   hx = -i cos(theta_jn) * h0,
 *     h0(f_k) = A(f_k) exp(-i Psi(f_k)) for f_lo <= f_k <= f_top(b), zero elsewhere (bin 0 and the
 *     Nyquist bin are always zero);  f_top = min(f_ISCO, f_hi) for TaylorF2, min(0.2/M, f_hi) for
 *     IMRPhenomD.  Phase is accumulated in fp64, amplitude in fp32.
 *   params [batch, 11] fp64;  hp, hc [batch, K, 2] fp32;  flags [batch] int32 or NULL. */
int amplfi_waveform_fd(const amplfi_plan* plan, int approximant, int batch, const double* params,
                       double f_lo, double f_hi, float* hp, float* hc, int* flags, void* stream);

/* a-2, a-3 Projection ("antenna response ... on-the-fly on the GPU"):
 *     h_d(f_k) = (F+_d h+ + Fx_d hx) exp(-2 pi i f_k dt_d),
 * F+, Fx the antenna patterns of detector d for (ra, dec, psi) at Greenwich sidereal angle gmst and
 * dt_d the arrival-time offset of detector d relative to the geocentre (computed in fp64).
 *   hp, hc [batch, K, 2];  h_det [batch, n_det, K, 2] fp32;
 *   resp NULL or [batch, n_det, 3] fp64 receiving (F+, Fx, dt).
 * hp/hc/h_det may be NULL if only resp is wanted (then resp must not be NULL). */
int amplfi_project(const amplfi_plan* plan, int batch, const double* params, double gmst,
                   const float* hp, const float* hc, float* h_det, double* resp, void* stream);

/* a-4 Welch PSD ("power spectra estimation"; "The power spectra is fit to
 * this background chunk"): per detector, segments of nperseg samples stepping by nperseg - noverlap
 * (full segments only), optional mean removal, periodic Hann window, |FFT|^2, mean over segments,
 * one-sided density.
 *   bg fp32 strain: detector d's n_bg samples start at bg + d * row_stride (row_stride in elements,
 *   >= n_bg; pass n_bg for a dense [n_det, n_bg] array, or the strip length to use a window of the
 *   GPU-resident strip in place);  noverlap in [0, nperseg);  detrend 0 none / 1 constant;
 *   average 0: mean over segments.  average 1: per-bin median over segments divided by the
 *   median-to-mean ratio of nseg exponentially distributed values (the middle order statistic of n unit
 *   exponentials has expectation sum_{j=n-k+1}^{n} 1/j; two middle ones averaged for even nseg), which is
 *   robust against loud transients in the background;  psd [n_det, nperseg/2+1] fp32 receives S * 2^140.
 * Deterministic (fixed summation order; ties in the median broken by segment index).  Backgrounds of more than 256
 * segments (the paper fits the PSD to a quarter-day chunk) are processed in groups of 256 whose sums are
 * added in order (mean only; the median of more than 256 segments returns AMPLFI_ERR_UNSUPPORTED_SIZE). */
int amplfi_psd_welch(const amplfi_plan* plan, const float* bg, long n_bg, long row_stride, int noverlap,
                     int detrend, int average, float* psd, void* stream);

/* The same estimate (mean over segments) for callers that may not allocate device memory: code under CUDA graph
 * capture, serving loops, harnesses that forbid cudaMalloc.  It needs no plan and calls no cudaMalloc, cudaFree or
 * allocating library routine: the per-segment periodograms go to a static device array of
 * AMPLFI_NOALLOC_WELCH_FLOATS floats (4 MiB, held by every GPU that loads the library until the process exits).
 *   bg, n_bg, row_stride, noverlap, detrend, psd as above;  n_det in [1, 3];  fs in Hz;  nperseg a power of two in
 *   [2^10, 2^15];  stream: the cudaStream_t of the launches.
 * Limit: n_det * nseg * (nperseg/2 + 1) <= AMPLFI_NOALLOC_WELCH_FLOATS, nseg = (n_bg - nperseg)/(nperseg - noverlap) + 1
 * (e.g. 3 detectors x 63 segments of 8192 samples); beyond it the call returns AMPLFI_ERR_UNSUPPORTED_SIZE and launches
 * nothing.  All calls share the one array: calls that overlap on the GPU (other streams, other threads) race on it and
 * must be serialised by the caller.  The array keeps the previous call's contents; every value that is read is written
 * first in the same call, so nothing needs clearing.  Results are bit-identical to amplfi_psd_welch(average = 0). */
#define AMPLFI_NOALLOC_WELCH_FLOATS (1 << 20)
int amplfi_psd_welch_noalloc(const float* bg, long n_bg, long row_stride, int n_det, double fs, int nperseg,
                             int noverlap, int detrend, float* psd, void* stream);

/* a-5 .. a-9 Gather + inject + whiten ("N small background chunks ... are lazily loaded";
 * PAPER.md:105 "We then inject the signals into the background chunks ... We whiten the batch using the
 * estimated power spectra"):
 *     out[b,d,:] = irfft( ( rfft(x[b,d,:]) + fs * h_d[b,:] ) * w_d ),
 *     w_d[k] = sqrt(2 / (fs * S_d(f_k))) for f_lo <= f_k <= f_hi, 0 elsewhere.
 *   noise    offsets == NULL: dense [batch, n_det, n] fp32.
 *            offsets != NULL: strip [n_det, strip_len] fp32 and x[b,d,:] = strip[d, offsets[b,d] : +n];
 *            offsets [batch, n_det] int64, each in [0, strip_len - n] (checked on the device: an
 *            out-of-range offset yields an all-NaN row, never an out-of-bounds read).
 *   h_det    [batch, n_det, K, 2] fp32 to inject a caller-supplied projected waveform, or NULL.
 *   params   used when h_det == NULL: [batch, 11] fp64 -> the waveform is generated, projected and
 *            injected inside the call (fused path; `approximant`, `gmst` as above; the waveform band is
 *            the same [f_lo, f_hi]).  h_det == NULL and params == NULL: whiten only.
 *   psd      [n_det, n_psd] fp32, S * 2^140; n_psd == K, or n_psd == (n/r)/2+1 for an integer r >= 1, in
 *            which case S is linearly interpolated in frequency onto the segment grid.
 *   out      [batch, n_det, n] fp32.
 * batch <= the plan's max_batch.  n = 2^16 and 2^17 run as a cluster of two / four thread blocks sharing the transform
 * through distributed shared memory; n >= 2^18 runs as a four-step transform around rows of 16384 complex points, the
 * rows of a chunk of segments staying in L2 (three launches per chunk). */
int amplfi_inject_whiten(const amplfi_plan* plan, int batch, const float* noise, const long* offsets,
                         long strip_len, const float* h_det, int approximant, const double* params,
                         double gmst, const float* psd, int n_psd, double f_lo, double f_hi,
                         float* out, void* stream);

/* Two data views (d, d') of the self-supervised pre-training (Figure 2: "the same background strain
 * with a time-shifted signal injected, the parameters of which are otherwise the same ... random up to 1s";
 * PAPER.md:117 "all signal parameters being the same except the time of arrival"):
 *     out  = amplfi_inject_whiten(fused) with params,
 *     out2 = the same with t_c replaced by t_c + t_shift[b]  (same noise segment, same PSD).
 * The per-sample coefficients and the h0 spectrum are computed once; the second view only changes the
 * linear phase exp(-2 pi i f_k (dt_d + t_shift[b])), accumulated in fp64.
 *   t_shift [batch] fp64 seconds;  out, out2 [batch, n_det, n] fp32;  other arguments as amplfi_inject_whiten
 *   (fused form: params must not be NULL). */
int amplfi_inject_whiten_views(const amplfi_plan* plan, int batch, const float* noise, const long* offsets,
                               long strip_len, int approximant, const double* params, const double* t_shift,
                               double gmst, const float* psd, int n_psd, double f_lo, double f_hi, float* out,
                               float* out2, void* stream);

/* Time-domain polarisations on the segment grid t_j = j / fs (Figure 1 shows the "time-domain
 * IMRPhenomD"): the inverse Fourier integral of the frequency-domain model sampled on the grid,
 *     h(t_j) = fs * irfft(h~)[j]      (circular on the segment; the band is cut sharply at f_lo and f_top),
 * computed by the inverse half of the segment transform without materialising h+~, hx~.
 *   params [batch, 11] fp64;  h_t [batch, 2, n] fp32 strain: row 0 = h+, row 1 = hx;  flags [batch] or NULL. */
int amplfi_waveform_td(const amplfi_plan* plan, int approximant, int batch, const double* params, double f_lo,
                       double f_hi, float* h_t, int* flags, void* stream);

/* amplfi_inject_whiten with the whitening filter truncated in time (the practice of the
 * library the paper delegates whitening to; reading R-I8):
 *   1. w[k] = sqrt(2/(fs S(f_k))) in [f_lo, f_hi], 0 outside;  2. q = irfft(w) (real, even);
 *   3. q'[j] = q[j] (1 + cos(2 pi m / ntaps))/2 for m = min(j, n-j) < ntaps/2, else 0, ntaps = fduration * fs;
 *   4. W' = rfft(q');  out = irfft((rfft(x) + fs h_d) W').
 * With crop = 1 the first and last ntaps/2 samples of every row, which the circular convolution contaminates
 * with data from the other end of the segment, are not written: out is [batch, n_det, n - ntaps] and equals
 * the linear convolution of the data with the ntaps-long filter.  crop = 0: out is [batch, n_det, n].
 *   fduration * fs must be a multiple of 4 in [4, n] (n - ntaps > 0 with crop);  other arguments as
 *   amplfi_inject_whiten. */
int amplfi_inject_whiten_fir(const amplfi_plan* plan, int batch, const float* noise, const long* offsets,
                             long strip_len, const float* h_det, int approximant, const double* params,
                             double gmst, const float* psd, int n_psd, double f_lo, double f_hi, double fduration,
                             int crop, float* out, void* stream);

/* One whole data-generation step (PSD fit to the background, waveforms generated on the
 * GPU, projected, injected into lazily loaded background chunks, batch whitened) = amplfi_psd_welch followed
 * by the fused amplfi_inject_whiten (h_det == NULL, params != NULL), with identical results.  The PSD chain
 * (Welch, filter) and the waveform chain (per-sample coefficients, h0 spectra) do not depend on each other, so
 * they run concurrently: the PSD chain on a stream owned by the plan, forked from and joined back into
 * `stream` with events; everything is ordered after prior work on `stream` and complete (in stream order)
 * when the call's last kernel on `stream` is.
 *   bg, n_bg, row_stride, noverlap, detrend as in amplfi_psd_welch;  psd [n_det, nperseg/2+1] receives the
 *   estimate;  noise, offsets, strip_len, approximant, params (not NULL), gmst, f_lo, f_hi, out as in
 *   amplfi_inject_whiten. */
int amplfi_assemble_batch(const amplfi_plan* plan, int batch, const float* bg, long n_bg, long row_stride,
                          int noverlap, int detrend, float* psd, const float* noise, const long* offsets,
                          long strip_len, int approximant, const double* params, double gmst, double f_lo,
                          double f_hi, float* out, void* stream);

/* Device timing of the dominant kernel (the fused inject+whiten kernel).  With timing enabled every
 * amplfi_inject_whiten call brackets that kernel with CUDA events recorded on the caller's stream (up to
 * 512 calls are kept; enabling resets the list).  amplfi_plan_kernel_times waits for the recorded events
 * and writes up to `max` durations in milliseconds to the HOST array ms; returns the number written, or a
 * negative error. */
int amplfi_plan_set_timing(amplfi_plan* plan, int enable);
int amplfi_plan_kernel_times(amplfi_plan* plan, float* ms, int max);

/* Measured fp32 arithmetic ceiling of the current device: runs a register-resident loop of packed fp32x2 FMAs
 * (2 lane-operations per thread-instruction) on every SM and writes the achieved fp32 lane-operations per second
 * to the HOST double *lane_ops_per_s.  This is the denominator of the second roofline bench.py reports for the
 * fused kernel, whose FFT butterflies are bound by the fp32 pipe rather than by HBM.
 * Synchronises the device; not part of the hot path. */
int amplfi_probe_fp32_pipe(double* lane_ops_per_s);

/* Number of kernel launches the library has enqueued since it was loaded (all plans, all threads).
 * bench.py reports the difference across its timed region as "gpu_launches". */
long amplfi_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* AMPLFI_H */
