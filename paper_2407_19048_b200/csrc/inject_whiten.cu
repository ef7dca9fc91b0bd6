// inject_whiten.cu -- the fused gather -> real FFT -> inject -> whiten/band-limit -> inverse real FFT kernel.
// PAPER.md:103 (background chunks "lazily loaded" from the GPU-resident strip), PAPER.md:105 ("inject the
// signals into the background chunks ... whiten the batch using the estimated power spectra").
//
// One CTA per (sample, detector) segment.  The segment lives in shared memory between the FFT passes and
// in registers during the per-bin work; HBM sees 4 B/sample in and 4 B/sample out (plus the L2-resident
// filter and, on the fused path, the per-sample h0 spectrum shared by the detectors of a sample).
#include "amplfi_internal.h"
#include "fft_core.cuh"
#include "spec_layout.cuh"
#include "waveform.cuh"

namespace amplfi {

// ---- whitening filter on the segment grid: w[k] = sqrt(2/(fs S)) / (2N) inside the band, else 0 ----
// psd holds S * 2^140, so sqrt(2/(fs S)) = 2^70 * rsqrt(fs * psd / 2).
__global__ void filter_kernel(const float* __restrict__ psd, int n_psd, int n_bins, int ratio, float fs, float norm,
                              int k_lo, int k_hi, float* __restrict__ filt, int filt_stride, float* __restrict__ filt_slots,
                              int kl) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int d = blockIdx.y;
    if (k >= filt_stride) return;
    float w = 0.f;
    if (k >= k_lo && k <= k_hi && k < n_bins) {
        const float* s = psd + (size_t)d * n_psd;
        float sv;
        if (ratio == 1) {
            sv = s[k];
        } else {
            int i0 = k / ratio;
            if (i0 > n_psd - 2) i0 = n_psd - 2;
            const float t = (float)(k - i0 * ratio) / (float)ratio;
            sv = (1.0f - t) * s[i0] + t * s[i0 + 1];
        }
        w = rsqrtf(0.5f * fs * sv) * norm;
    }
    filt[(size_t)d * filt_stride + k] = w;
    if (filt_slots != nullptr && k < 16 * kl) filt_slots[(size_t)d * slot::filt_row(kl) + slot::filt_index(kl, k)] = w;
}

int launch_filter(const amplfi_plan* p, const float* psd, int n_psd, double f_lo, double f_hi, cudaStream_t st) {
    const int ratio = (p->n / 2) / (n_psd - 1);
    long k_lo = (long)ceil(f_lo * p->t_seg);
    while ((double)(k_lo - 1) / p->t_seg >= f_lo) --k_lo;
    while ((double)k_lo / p->t_seg < f_lo) ++k_lo;
    long k_hi = (long)floor(f_hi * p->t_seg);
    while ((double)(k_hi + 1) / p->t_seg <= f_hi) ++k_hi;
    while (k_hi >= 0 && (double)k_hi / p->t_seg > f_hi) --k_hi;
    if (k_lo < 0) k_lo = 0;
    if (k_hi > p->n_bins - 1) k_hi = p->n_bins - 1;
    const float norm = (float)(1180591620717411303424.0 / (2.0 * (double)p->n));      // 2^70 / (2N)
    dim3 grid((p->filt_stride + 255) / 256, p->n_det);
    filter_kernel<<<grid, 256, 0, st>>>(psd, n_psd, p->n_bins, ratio, (float)p->fs, norm, (int)k_lo, (int)k_hi, p->filt,
                                        p->filt_stride, p->filt_slots, p->n / 32);
    count_launch();
    return check_launch("filter_kernel");
}

// ---- time-truncated whitening filter (reading R-I8) ----
// The filter w (real, on the segment grid) has a real even impulse response q = irfft(w); q is tapered to ntaps samples
// around lag 0 with a Hann window and transformed back.  Both transforms are INVERSE real transforms of a real "spectrum"
// (for a real even sequence the forward transform equals n times the inverse one), so they run through the inverse half
// of the segment kernel (noise == nullptr, MODE_HDET) with one unit per detector:
//   time = fs * irfft(spec)   (two_fs * spec * 1/(2n), unnormalised inverse)
__global__ void fir_real_to_spec_kernel(const float* __restrict__ src, int src_stride, int n_bins, float mul, int ntaps,
                                        float2* __restrict__ spec) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int d = blockIdx.y;
    if (k >= n_bins) return;
    float v = src[(size_t)d * src_stride + k] * mul;
    if (ntaps > 0) {                                       // Hann taper centred on lag 0; lags k <= n/2 only (q is even)
        v = (2 * k < ntaps) ? v * (0.5f + 0.5f * cospif(2.0f * (float)k / (float)ntaps)) : 0.f;
    }
    spec[(size_t)d * n_bins + k] = make_float2(v, 0.f);
}

__global__ void fir_time_to_filt_kernel(const float* __restrict__ time, int n, int n_bins, float mul, float* __restrict__ filt,
                                        int filt_stride, float* __restrict__ filt_slots, int kl) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int d = blockIdx.y;
    if (k >= filt_stride) return;
    const float w = k < n_bins ? time[(size_t)d * n + k] * mul : 0.f;
    filt[(size_t)d * filt_stride + k] = w;
    if (filt_slots != nullptr && k < 16 * kl) filt_slots[(size_t)d * slot::filt_row(kl) + slot::filt_index(kl, k)] = w;
}

// plan->filt (already holding the band-limited filter of launch_filter) is replaced by its time-truncated version.
int launch_fir_truncate(const amplfi_plan* p, double fduration, cudaStream_t st) {
    const int ntaps = (int)llrint(fduration * p->fs);
    const int nb = p->n_bins;
    const float inv_fs = (float)(1.0 / p->fs);
    dim3 gb((nb + 255) / 256, p->n_det), gf((p->filt_stride + 255) / 256, p->n_det);
    IwOpts o;
    o.n_det = 1; o.resp = nullptr; o.filt = p->filt_flat; o.filt_stride = 0; o.crop = 0; o.phase64 = 0; o.out2 = nullptr; o.t_shift = nullptr;
    // q = irfft(w): time = fs q
    fir_real_to_spec_kernel<<<gb, 256, 0, st>>>(p->filt, p->filt_stride, nb, 1.0f, 0, p->fir_spec);
    count_launch();
    int rc = launch_inject_whiten(p, p->n_det, nullptr, nullptr, 0, reinterpret_cast<const float*>(p->fir_spec), 0,
                                  p->fir_time, st, &o);
    if (rc) return rc;
    // q' = taper(q) on lags 0 .. n/2; W' = rfft(q') = n irfft(q'[0 .. n/2]): time = fs W' / n
    fir_real_to_spec_kernel<<<gb, 256, 0, st>>>(p->fir_time, p->n, nb, inv_fs, ntaps, p->fir_spec);
    count_launch();
    rc = launch_inject_whiten(p, p->n_det, nullptr, nullptr, 0, reinterpret_cast<const float*>(p->fir_spec), 0, p->fir_time,
                              st, &o);
    if (rc) return rc;
    fir_time_to_filt_kernel<<<gf, 256, 0, st>>>(p->fir_time, p->n, nb, (float)((double)p->n / p->fs), p->filt, p->filt_stride, p->filt_slots, p->n / 32);
    count_launch();
    return check_launch("fir_truncate");
}

template <int LOGM, int MODE>
__global__ void __launch_bounds__(Fft<LOGM>::T) inject_whiten_kernel(const IwArgs a) {
    using F = Fft<LOGM>;
    constexpr int M = F::M, N = 2 * M, K = M + 1, RA = F::RA, RC = F::RC, T = F::T, LB = F::LB;
    extern __shared__ float2 sm[];
    const int unit = blockIdx.x, tid = threadIdx.x;
    const int b = unit / a.n_det, d = unit - b * a.n_det;

    // ---- a-5 gather ----
    const float* x = nullptr;
    const int n_out = N - 2 * a.crop;
    float* out = a.out + (size_t)unit * n_out;
    if (a.noise == nullptr) {
        // inverse-only launch: no data, the spectrum starts at zero
    } else if (a.offsets != nullptr) {
        const long off = a.offsets[unit];
        if (off < 0 || off + N > a.strip_len) {            // never read out of bounds: poison the row instead
            const float qnan = __int_as_float(0x7fc00000);
            for (int i = tid; i < n_out; i += T) out[i] = qnan;
            return;
        }
        x = a.noise + (size_t)d * a.strip_len + off;
    } else {
        x = a.noise + (size_t)unit * N;
    }
    const bool aligned8 = ((reinterpret_cast<size_t>(x) & 7) == 0);
    int klow_a, klow_b;
    pass_c_klow<LOGM>(tid, klow_a, klow_b);
    float2 va[RC], vb[RC];

    // ---- a-6 forward real FFT (packed as M complex points) ----
    if (x != nullptr) {
      {
        float2 v[F::NA][RA];
        if (aligned8) {
            const float2* x2 = reinterpret_cast<const float2*>(x);
#pragma unroll
            for (int i = 0; i < F::NA; ++i)
#pragma unroll
                for (int nA = 0; nA < RA; ++nA) v[i][nA] = __ldcs(x2 + nA * LB + tid + i * T);
        } else {
#pragma unroll
            for (int i = 0; i < F::NA; ++i)
#pragma unroll
                for (int nA = 0; nA < RA; ++nA) {
                    const int m = nA * LB + tid + i * T;
                    v[i][nA] = make_float2(__ldg(x + 2 * m), __ldg(x + 2 * m + 1));
                }
        }
#pragma unroll
        for (int i = 0; i < F::NA; ++i) F::pass_a_fwd(v[i], tid + i * T, sm);
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < F::NB; ++i) F::pass_b_fwd(tid + i * T, sm);
      __syncthreads();
      F::pass_c_fwd(klow_a, va, sm);
      F::pass_c_fwd(klow_b, vb, sm);
    } else {
#pragma unroll
      for (int i = 0; i < RC; ++i) va[i] = vb[i] = make_float2(0.f, 0.f);
    }

    // ---- a-7 inject, a-8 whiten + band-limit (registers) ----
    const float* filt = a.filt + (size_t)d * a.filt_stride;
    const float2* hsrc = nullptr;
    int w_lo = 1, w_hi = 0;
    float cre = 0.f, cim = 0.f;
    double delta = 0.0;
    if (MODE == MODE_HDET) hsrc = a.h_det + (size_t)unit * K;
    if (MODE == MODE_FUSED) {
        const WfCoef* c = a.coef + b;
        hsrc = a.h0 + (size_t)b * K;
        if (c->valid) { w_lo = c->k_lo; w_hi = c->k_hi; }
        const DetResp r = a.resp[unit];
        cre = (float)r.fp * c->pol_p;                       // C = F+ (1+cos^2 i)/2 - i Fx cos i
        cim = -(float)r.fc * c->pol_c;
        delta = r.dt * (double)a.inv_tseg;                   // turns per bin (fp64: the second view's dt reaches 1 s)
    }
    auto inject = [&](int k, float2& x2) {
        if (MODE == MODE_HDET) {
            const float2 h = __ldg(hsrc + k);
            x2.x = fmaf(a.two_fs, h.x, x2.x);
            x2.y = fmaf(a.two_fs, h.y, x2.y);
        } else if (MODE == MODE_FUSED) {
            if (k >= w_lo && k <= w_hi) {
                const float2 h = __ldg(hsrc + k);
                double td = (double)k * delta;
                td -= rint(td);
                float s, co;
                __sincosf((float)td * -6.283185307179586f, &s, &co);      // exp(-2 pi i k dt / T)
                const float2 cp = make_float2(cre * co - cim * s, cre * s + cim * co);
                x2.x += h.x * cp.x - h.y * cp.y;
                x2.y += h.x * cp.y + h.y * cp.x;
            }
        }
    };
    for_each_bin_pair<LOGM>(
        tid, va, vb,
        [&](int k, float2& za, float2& zb) {
            const float2 w = twiddle<N>(k);
            float2 xa, xb;
            split_pair(za, zb, w, xa, xb);
            inject(k, xa);
            inject(M - k, xb);
            const float fa = __ldg(filt + k), fb = __ldg(filt + M - k);
            xa.x *= fa; xa.y *= fa; xb.x *= fb; xb.y *= fb;
            merge_pair(xa, xb, w, za, zb);
        },
        [&](int k, float2& z) {
            const float2 w = twiddle<N>(k);
            float2 xa, xb, z2;
            split_pair(z, z, w, xa, xb);
            inject(k, xa);
            const float fa = __ldg(filt + k);
            xa.x *= fa; xa.y *= fa;
            merge_pair(xa, xa, w, z, z2);
        },
        [&](float2& z) {
            float x0 = 2.0f * (z.x + z.y), xm = 2.0f * (z.x - z.y);       // 2 X[0], 2 X[M] (real)
            if (MODE == MODE_HDET) {
                x0 = fmaf(a.two_fs, __ldg(hsrc).x, x0);
                xm = fmaf(a.two_fs, __ldg(hsrc + M).x, xm);
            }
            const float y0 = x0 * __ldg(filt), ym = xm * __ldg(filt + M);
            z = make_float2(y0 + ym, y0 - ym);                            // 4 Z'[0]
        });

    // ---- a-9 inverse real FFT and store ----
    F::pass_c_inv(klow_a, va, sm);
    F::pass_c_inv(klow_b, vb, sm);
    __syncthreads();
#pragma unroll
    for (int i = 0; i < F::NB; ++i) F::pass_b_inv(tid + i * T, sm);
    __syncthreads();
    float2* out2 = reinterpret_cast<float2*>(out);
#pragma unroll
    for (int i = 0; i < F::NA; ++i) {
        float2 v[RA];
        F::pass_a_inv(v, tid + i * T, sm);
        if (a.crop == 0) {
#pragma unroll
            for (int nA = 0; nA < RA; ++nA) __stcs(out2 + nA * LB + tid + i * T, v[nA]);
        } else {
            const int c2 = a.crop >> 1;                      // crop is even: whole float2 pairs
#pragma unroll
            for (int nA = 0; nA < RA; ++nA) {
                const int m = nA * LB + tid + i * T;
                if (m >= c2 && m < M - c2) __stcs(out2 + m - c2, v[nA]);
            }
        }
    }
}

template <int LOGM, int MODE>
static int launch_iw_t(const IwArgs& a, int units, cudaStream_t st) {
    using F = Fft<LOGM>;
    static std::atomic<unsigned> attr_done{0};
    const int rc = ensure_dynamic_smem(inject_whiten_kernel<LOGM, MODE>, (int)F::SMEM_BYTES, attr_done);
    if (rc) return rc;
    inject_whiten_kernel<LOGM, MODE><<<units, F::T, F::SMEM_BYTES, st>>>(a);
    count_launch();
    return check_launch("inject_whiten_kernel");
}

template <int LOGM>
static int launch_iw_mode(const IwArgs& a, int mode, int units, cudaStream_t st) {
    switch (mode) {
        case MODE_NONE: return launch_iw_t<LOGM, MODE_NONE>(a, units, st);
        case MODE_HDET: return launch_iw_t<LOGM, MODE_HDET>(a, units, st);
        default: return launch_iw_t<LOGM, MODE_FUSED>(a, units, st);
    }
}

int launch_inject_whiten(const amplfi_plan* p, int batch, const float* noise, const long* offsets,
                         long strip_len, const float* h_det, int fused, float* out, cudaStream_t st,
                         const IwOpts* opts) {
    IwArgs a;
    a.noise = noise; a.offsets = offsets; a.strip_len = strip_len;
    a.h_det = reinterpret_cast<const float2*>(h_det);
    a.h0 = p->h0; a.coef = p->coef; a.resp = p->resp; a.filt = p->filt; a.filt_stride = p->filt_stride; a.out = out;
    a.filt_slots = p->filt_slots;
    a.crop = 0; a.phase64 = 0; a.out2 = nullptr; a.t_shift = nullptr;
    a.n_det = p->n_det; a.two_fs = (float)(2.0 * p->fs); a.inv_tseg = (float)(1.0 / p->t_seg);
    a.prefetch_ahead = (p->logm >= 11 && p->logm <= 14 ? 1 : 2) * p->sm_count * (8192 / (p->n / 2 < 8192 ? p->n / 2 : 8192));   // one wave ahead
    if (p->logm >= 15) a.prefetch_ahead = p->sm_count >> (p->logm - 14);      // one cluster of 2 / 4 CTAs per unit
    if (opts != nullptr) {
        a.n_det = opts->n_det;
        if (opts->resp != nullptr) a.resp = opts->resp;
        if (opts->filt != nullptr) { a.filt = opts->filt; a.filt_stride = opts->filt_stride; a.filt_slots = opts->filt; }
        a.crop = opts->crop; a.phase64 = opts->phase64;
        if (p->logm >= 11 && p->logm <= 13) { a.out2 = opts->out2; a.t_shift = opts->t_shift; }
    }
    const int mode = h_det != nullptr ? MODE_HDET : (fused ? MODE_FUSED : MODE_NONE);
    const int units = batch * a.n_det;
    switch (p->logm) {
        case 9: return launch_iw_mode<9>(a, mode, units, st);
        case 10: return launch_iw_mode<10>(a, mode, units, st);
        case 11: case 12: case 13: case 14: case 15: case 16: return launch_iw3(a, p->logm, mode, units, st);
        case 17: case 18: case 19: return launch_inject_whiten_long(p, a, mode, units, st);
        default:
            set_error("amplfi_inject_whiten: segment length %d not supported by this build", p->n);
            return AMPLFI_ERR_UNSUPPORTED_SIZE;
    }
}

}  // namespace amplfi
