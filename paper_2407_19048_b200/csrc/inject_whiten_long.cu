// inject_whiten_long.cu -- gather -> FFT -> inject -> whiten -> iFFT for n = 2^16 .. 2^20 (config c4: 16 s at 4096 Hz;
// the minutes-long segments of binary-neutron-star signals).
// PAPER.md:103, :105 (same step as inject_whiten.cu); "the signal duration can be O(min) ... This makes the
// input arrays larger by an order of magnitude".
//
// A segment longer than 32768 samples does not fit one CTA's shared memory, so the transform is decimated in time by
// R = n / 32768 (2 .. 32) around the single-CTA 32768-sample real transform of fft_core.cuh, the intermediate spectra
// staying in L2:
//   x_r[m] = x[R m + r], r < R, m < ns = 32768              R real sequences with spectra X_r[k], k <= ns/2
//   X[k] = sum_r w_n^(r k) X_r[k mod ns], 0 <= k <= n/2,     X_r[ns - k] = conj(X_r[k])
// then the pointwise stage (inject, whiten, band-limit) on X, the same sum backwards into the sub-spectra Y_r of the
// output, and y[R m + r] = irfft(Y_r)[m].  Three kernels per chunk of units: sub-spectra (one CTA per unit and r), the
// element-wise stage (one thread per sub-spectrum bin, R bins of the full spectrum each), inverse sub-transforms.  A
// chunk's spectra (n * 4 B per unit) are sized to stay resident in the 126 MB L2, so HBM sees the algorithmic 8 B per
// sample.  First correct version: strided scalar gathers, an O(R) sum per bin instead of a radix-R butterfly.
#include "amplfi_internal.h"
#include "fft_core.cuh"
#include "waveform.cuh"

namespace amplfi {

constexpr int LONG_LOGM = 14;                       // sub-transform: 16384 complex = 32768 real samples
constexpr int LONG_KS = (1 << LONG_LOGM) + 1;        // bins of a sub-spectrum
constexpr int LONG_KS_STRIDE = LONG_KS + 7;          // row stride in float2 (multiple of 8)
constexpr int LONG_NS = 2 << LONG_LOGM;              // samples of a sub-sequence: 32768

struct LongArgs {
    const float* noise;
    const long* offsets;
    long strip_len;
    float2* spec;             // [chunk, 2, LONG_KS_STRIDE]
    float* out;
    int n_det;
    int unit0;                // first unit of the chunk
    int n_full;               // n
    int rdec;                 // R = n / 32768
    int crop;                 // samples dropped at each end of an output row (even)
};

// DIR = 0: x[R m + r] -> 2 X_r[k] (spectrum to scratch).  DIR = 1: spectrum from scratch -> y[R m + r].
template <int DIR>
__global__ void __launch_bounds__(Fft<LONG_LOGM>::T) long_sub_kernel(const LongArgs a) {
    constexpr int LOGM = LONG_LOGM;
    using F = Fft<LOGM>;
    constexpr int M = F::M, N = 2 * M, RA = F::RA, RC = F::RC, T = F::T, LB = F::LB;
    static_assert(F::NA == 1 && F::NB == 1, "long_sub_kernel assumes one butterfly per thread per pass");
    extern __shared__ float2 sm[];
    const int tid = threadIdx.x;
    const int R = a.rdec;
    const int lu = blockIdx.x / R, par = blockIdx.x - lu * R;
    const int unit = a.unit0 + lu;
    const int d = unit % a.n_det;
    float2* spec = a.spec + ((size_t)lu * R + par) * LONG_KS_STRIDE;
    const int n_out = a.n_full - 2 * a.crop;
    float* out = a.out + (size_t)unit * n_out;

    const float* x = nullptr;
    if (a.offsets != nullptr) {
        const long off = a.offsets[unit];
        if (off < 0 || off + a.n_full > a.strip_len) {      // never read out of bounds: poison the row instead
            if (DIR == 1) {
                const float qnan = __int_as_float(0x7fc00000);
                for (long i = tid; R * i + par < n_out; i += T) out[R * i + par] = qnan;
            }
            return;
        }
        x = a.noise + (size_t)d * a.strip_len + off;
    } else {
        x = a.noise + (size_t)unit * a.n_full;
    }

    int klow_a, klow_b;
    pass_c_klow<LOGM>(tid, klow_a, klow_b);
    float2 va[RC], vb[RC];

    if (DIR == 0) {
        {
            float2 v[RA];
            // packed point m of the sub-sequence: (x_r[2m], x_r[2m+1]) = (x[2 R m + r], x[2 R m + R + r])
#pragma unroll
            for (int nA = 0; nA < RA; ++nA) {
                const size_t m = (size_t)(nA * LB + tid);
                v[nA] = make_float2(__ldg(x + 2 * R * m + par), __ldg(x + 2 * R * m + R + par));
            }
            F::pass_a_fwd(v, tid, sm);
        }
        __syncthreads();
        F::pass_b_fwd(tid, sm);
        __syncthreads();
        F::pass_c_fwd(klow_a, va, sm);
        F::pass_c_fwd(klow_b, vb, sm);
        for_each_bin_pair<LOGM>(
            tid, va, vb,
            [&](int k, float2& za, float2& zb) {
                float2 xa, xb;
                split_pair(za, zb, twiddle<N>(k), xa, xb);
                spec[k] = xa;
                spec[M - k] = xb;
            },
            [&](int k, float2& z) {
                float2 xa, xb;
                split_pair(z, z, twiddle<N>(k), xa, xb);
                spec[k] = xa;
            },
            [&](float2& z) {
                spec[0] = make_float2(2.0f * (z.x + z.y), 0.f);
                spec[M] = make_float2(2.0f * (z.x - z.y), 0.f);
            });
    } else {
        for_each_bin_pair<LOGM>(
            tid, va, vb,
            [&](int k, float2& za, float2& zb) {
                const float2 xa = spec[k], xb = spec[M - k];
                merge_pair(xa, xb, twiddle<N>(k), za, zb);
            },
            [&](int k, float2& z) {
                const float2 xa = spec[k];
                float2 z2;
                merge_pair(xa, xa, twiddle<N>(k), z, z2);
            },
            [&](float2& z) {
                const float y0 = spec[0].x, ym = spec[M].x;
                z = make_float2(y0 + ym, y0 - ym);
            });
        F::pass_c_inv(klow_a, va, sm);
        F::pass_c_inv(klow_b, vb, sm);
        __syncthreads();
        F::pass_b_inv(tid, sm);
        __syncthreads();
        float2 v[RA];
        F::pass_a_inv(v, tid, sm);
#pragma unroll
        for (int nA = 0; nA < RA; ++nA) {
            const long m = nA * LB + tid;
            const long j0 = 2 * R * m + par - a.crop, j1 = j0 + R;
            if (j0 >= 0 && j0 < n_out) out[j0] = v[nA].x;
            if (j1 >= 0 && j1 < n_out) out[j1] = v[nA].y;
        }
    }
}

struct LongPwArgs {
    float2* spec;
    const float2* h_det;      // MODE_HDET: [B, D, K]
    const float2* h0;         // MODE_FUSED: [B, K] (2 fs h0)
    const WfCoef* coef;
    const DetResp* resp;
    const float* filt;
    int filt_stride;
    int n_det;
    int unit0;
    float two_fs;
    double inv_tseg;
    int nofwd;                // no data: the sub-spectra are taken as zero (inverse-only launches)
};

// exp(-2 pi i num / den) for a power-of-two den <= 2^21: the argument is reduced exactly in integers to [-pi, pi) and
// evaluated with the fast sine/cosine (absolute error ~4e-7, as for the twiddles of the transforms themselves)
__device__ __forceinline__ float2 long_w(long num, int den) {
    int m = (int)(num & (long)(den - 1));
    if (m >= den / 2) m -= den;
    float s, c;
    __sincosf((float)m * (-6.283185307179586f / (float)den), &s, &c);
    return make_float2(c, s);
}

// One thread per sub-spectrum bin k0 in [0, ns/2] and the R bins of the full one-sided spectrum that depend on it:
//   family 0: k = k0 + j ns        (built from X_r[k0])
//   family 1: k = (j + 1) ns - k0  (built from conj X_r[k0]),   j < R/2.
// Folding back, Y_r[k0] = sum over the FULL Hermitian spectrum of Y[k0 + j ns] w_n^(-r (k0 + j ns)), j < R; the upper
// half enters through the mirrored bins, conj(Y[k]) w_n^(+r k) with k of family 1.  For 0 < k0 < ns/2 the R bins are
// distinct.  At k0 = 0 and k0 = ns/2 the two families name the same bins, each bin 0 < k < n/2 standing for itself and for
// its mirror (weight 2, real part) and the real bins k = 0 and k = n/2 for themselves only (weight 1).
template <int MODE, int R>
__global__ void __launch_bounds__(128) long_pointwise_kernel(const LongPwArgs a) {
    constexpr int KS = LONG_KS, NS = LONG_NS, NF = R * NS, MF = NF / 2, KF = MF + 1;     // MF = n/2
    const int k0 = blockIdx.x * blockDim.x + threadIdx.x;
    if (k0 >= KS) return;
    const int lu = blockIdx.y;
    const int unit = a.unit0 + lu;
    const int b = unit / a.n_det, d = unit - b * a.n_det;
    float2* sp = a.spec + (size_t)lu * R * LONG_KS_STRIDE + k0;
    const float* filt = a.filt + (size_t)d * a.filt_stride;

    const float2* hsrc = nullptr;
    int w_lo = 1, w_hi = 0;
    float cre = 0.f, cim = 0.f;
    double delta = 0.0;
    if (MODE == MODE_HDET) hsrc = a.h_det + (size_t)unit * KF;
    if (MODE == MODE_FUSED) {
        const WfCoef* c = a.coef + b;
        hsrc = a.h0 + (size_t)b * KF;
        if (c->valid) { w_lo = c->k_lo; w_hi = c->k_hi; }
        const DetResp r = a.resp[unit];
        cre = (float)r.fp * c->pol_p;                       // C = F+ (1+cos^2 i)/2 - i Fx cos i
        cim = -(float)r.fc * c->pol_c;
        delta = r.dt * a.inv_tseg;                          // turns per bin
    }
    // a-7, a-8 at full-spectrum bin k: y = (x + injection) * filter   (x holds 2 X[k])
    auto pointwise = [&](int k, float2 x) -> float2 {
        if (MODE == MODE_HDET) {
            const float2 h = __ldg(hsrc + k);
            x.x = fmaf(a.two_fs, h.x, x.x);
            x.y = fmaf(a.two_fs, h.y, x.y);
        } else if (MODE == MODE_FUSED) {
            if (k >= w_lo && k <= w_hi) {
                const float2 hv = __ldg(hsrc + k);
                double turns = (double)k * delta;
                turns -= rint(turns);
                float s, co;
                __sincosf((float)turns * -6.283185307179586f, &s, &co);   // exp(-2 pi i k dt / T), |turns| <= 1/2
                const float2 cp = make_float2(cre * co - cim * s, cre * s + cim * co);
                x.x += hv.x * cp.x - hv.y * cp.y;
                x.y += hv.x * cp.y + hv.y * cp.x;
            }
        }
        const float f = __ldg(filt + k);
        return make_float2(x.x * f, x.y * f);
    };

    float2 v[R], acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        v[r] = a.nofwd ? make_float2(0.f, 0.f) : sp[(size_t)r * LONG_KS_STRIDE];
        acc[r] = make_float2(0.f, 0.f);
    }
    const bool edge = (k0 == 0 || k0 == NS / 2);

#pragma unroll(R <= 4 ? 2 : 1)
    for (int fam = 0; fam < 2; ++fam) {
#pragma unroll(R <= 4 ? R / 2 : 1)
        for (int j = 0; j < R / 2; ++j) {
            const int k = fam == 0 ? k0 + j * NS : (j + 1) * NS - k0;
            if (fam == 1 && k0 == 0 && j < R / 2 - 1) continue;     // k = (j+1) ns: visited by family 0
            if (fam == 1 && k0 == NS / 2) continue;                 // k = j ns + ns/2: visited by family 0
            // X[k] = sum_r w_n^(r k) V_r,  V_r = X_r[k0] (family 0) or its conjugate (family 1)
            const float2 w1 = long_w((long)k, NF);
            float2 wr = make_float2(1.f, 0.f), x = make_float2(0.f, 0.f);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if ((r & 7) == 0 && r > 0) wr = long_w((long)r * k, NF);          // restart the recurrence every 8 steps
                const float2 vr = fam == 0 ? v[r] : make_float2(v[r].x, -v[r].y);
                x.x += vr.x * wr.x - vr.y * wr.y;
                x.y += vr.x * wr.y + vr.y * wr.x;
                wr = cmul(wr, w1);
            }
            float2 y = pointwise(k, x);
            const bool real_bin = (k == 0 || k == MF);              // DC / Nyquist of a real sequence
            if (real_bin) y.y = 0.f;
            const float wgt = (edge && !real_bin) ? 2.0f : 1.0f;
            // fold back: Y[k] w_n^(-r k) (family 0) or conj(Y[k]) w_n^(+r k) (family 1, the mirrored half)
            const float2 yy = fam == 0 ? make_float2(wgt * y.x, wgt * y.y) : make_float2(wgt * y.x, -wgt * y.y);
            const float2 u1 = fam == 0 ? make_float2(w1.x, -w1.y) : w1;
            float2 ur = make_float2(1.f, 0.f);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if ((r & 7) == 0 && r > 0) {
                    const float2 t = long_w((long)r * k, NF);
                    ur = fam == 0 ? make_float2(t.x, -t.y) : t;
                }
                acc[r].x += yy.x * ur.x - yy.y * ur.y;
                acc[r].y += yy.x * ur.y + yy.y * ur.x;
                ur = cmul(ur, u1);
            }
        }
    }
    // no 1/R here: the filter carries the 1/(2n) of the whole transform (the sub-transforms are unnormalised)
#pragma unroll
    for (int r = 0; r < R; ++r) sp[(size_t)r * LONG_KS_STRIDE] = make_float2(acc[r].x, edge ? 0.f : acc[r].y);
}

static int long_attr() {
    static std::atomic<unsigned> done0{0}, done1{0};
    const int rc = ensure_dynamic_smem(long_sub_kernel<0>, (int)Fft<LONG_LOGM>::SMEM_BYTES, done0);
    return rc ? rc : ensure_dynamic_smem(long_sub_kernel<1>, (int)Fft<LONG_LOGM>::SMEM_BYTES, done1);
}

size_t long_scratch_floats2(int chunk_units, int rdec) { return (size_t)chunk_units * rdec * LONG_KS_STRIDE; }

template <int R>
static void launch_long_pw(const LongPwArgs& w, int mode, int cu, cudaStream_t st) {
    dim3 grid((LONG_KS + 127) / 128, cu);
    switch (mode) {
        case MODE_NONE: long_pointwise_kernel<MODE_NONE, R><<<grid, 128, 0, st>>>(w); break;
        case MODE_HDET: long_pointwise_kernel<MODE_HDET, R><<<grid, 128, 0, st>>>(w); break;
        default: long_pointwise_kernel<MODE_FUSED, R><<<grid, 128, 0, st>>>(w); break;
    }
}

int launch_inject_whiten_long(const amplfi_plan* p, const IwArgs& ia, int mode, int units, cudaStream_t st) {
    int rc = long_attr();
    if (rc) return rc;
    using F = Fft<LONG_LOGM>;
    const bool nofwd = ia.noise == nullptr;
    const int R = p->n / LONG_NS;
    for (int u0 = 0; u0 < units; u0 += p->long_chunk) {
        const int cu = units - u0 < p->long_chunk ? units - u0 : p->long_chunk;
        LongArgs a;
        a.noise = ia.noise; a.offsets = nofwd ? nullptr : ia.offsets; a.strip_len = ia.strip_len; a.spec = p->long_spec;
        a.out = ia.out; a.n_det = ia.n_det; a.unit0 = u0; a.n_full = p->n; a.rdec = R; a.crop = ia.crop;
        if (!nofwd) { long_sub_kernel<0><<<R * cu, F::T, F::SMEM_BYTES, st>>>(a); count_launch(); }
        LongPwArgs w;
        w.spec = p->long_spec; w.h_det = ia.h_det; w.h0 = ia.h0; w.coef = ia.coef;
        w.resp = ia.resp; w.filt = ia.filt; w.filt_stride = ia.filt_stride; w.n_det = ia.n_det; w.unit0 = u0;
        w.two_fs = ia.two_fs; w.inv_tseg = 1.0 / p->t_seg; w.nofwd = nofwd ? 1 : 0;
        switch (R) {
            case 2: launch_long_pw<2>(w, mode, cu, st); break;
            case 4: launch_long_pw<4>(w, mode, cu, st); break;
            case 8: launch_long_pw<8>(w, mode, cu, st); break;
            case 16: launch_long_pw<16>(w, mode, cu, st); break;
            case 32: launch_long_pw<32>(w, mode, cu, st); break;
            default: set_error("inject_whiten_long: n = %d not supported", p->n); return AMPLFI_ERR_UNSUPPORTED_SIZE;
        }
        long_sub_kernel<1><<<R * cu, F::T, F::SMEM_BYTES, st>>>(a);
        count_launch(2);
    }
    return check_launch("inject_whiten_long");
}

}  // namespace amplfi
