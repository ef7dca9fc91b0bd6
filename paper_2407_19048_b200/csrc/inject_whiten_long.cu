// inject_whiten_long.cu -- gather -> FFT -> inject -> whiten -> iFFT for n = 65536 (config c4: 16 s at 4096 Hz).
// PAPER.md:103, :105 (same step as inject_whiten.cu); PAPER.md:212 notes that longer signals need longer arrays.
//
// 32768 complex points (256 KB) do not fit one CTA's shared memory, so the transform is decimated in time by two
// ("four-step" with the intermediate kept in L2):
//   xe[m] = x[2m], xo[m] = x[2m+1]                      two real sequences of 32768 samples
//   A = Xe[k], B = w_N^k Xo[k], 0 <= k <= 16384:         X[k] = A + B,  X[N/2 - k] = conj(A - B)
//   pointwise (inject, whiten, band-limit) on both bins, then with P = Y[k], Q = conj(Y[N/2 - k]):
//   Ye[k] = (P + Q)/2,  Yo[k] = conj(w_N^k) (P - Q)/2,   y[2m] = irfft(Ye)[m],  y[2m+1] = irfft(Yo)[m]
// Three kernels per chunk of units: sub-spectra (one CTA per unit and parity, the single-CTA 32768-sample transform
// of fft_core.cuh), the element-wise combine/pointwise/split, and the inverse sub-transforms.  A chunk's spectra
// (262 KB per unit) are sized to stay resident in the 126 MB L2, so HBM sees the algorithmic 8 B per sample.
#include "amplfi_internal.h"
#include "fft_core.cuh"
#include "waveform.cuh"

namespace amplfi {

constexpr int LONG_LOGM = 14;                       // sub-transform: 16384 complex = 32768 real samples
constexpr int LONG_KS = (1 << LONG_LOGM) + 1;        // bins of a sub-spectrum
constexpr int LONG_KS_STRIDE = LONG_KS + 7;          // row stride in float2 (multiple of 8)

struct LongArgs {
    const float* noise;
    const long* offsets;
    long strip_len;
    float2* spec;             // [chunk, 2, LONG_KS_STRIDE]
    float* out;
    int n_det;
    int unit0;                // first unit of the chunk
    int n_full;               // 65536
    int crop;                 // samples dropped at each end of an output row (even)
};

// DIR = 0: x[2m+p] -> 2 Xp[k] (spectrum to scratch).  DIR = 1: spectrum from scratch -> y[2m+p].
template <int DIR>
__global__ void __launch_bounds__(Fft<LONG_LOGM>::T) long_sub_kernel(const LongArgs a) {
    constexpr int LOGM = LONG_LOGM;
    using F = Fft<LOGM>;
    constexpr int M = F::M, N = 2 * M, RA = F::RA, RC = F::RC, T = F::T, LB = F::LB;
    static_assert(F::NA == 1 && F::NB == 1, "long_sub_kernel assumes one butterfly per thread per pass");
    extern __shared__ float2 sm[];
    const int tid = threadIdx.x;
    const int lu = blockIdx.x >> 1, par = blockIdx.x & 1;
    const int unit = a.unit0 + lu;
    const int d = unit % a.n_det;
    float2* spec = a.spec + ((size_t)lu * 2 + par) * LONG_KS_STRIDE;
    const int n_out = a.n_full - 2 * a.crop;
    float* out = a.out + (size_t)unit * n_out;

    const float* x = nullptr;
    if (a.offsets != nullptr) {
        const long off = a.offsets[unit];
        if (off < 0 || off + a.n_full > a.strip_len) {      // never read out of bounds: poison the row instead
            if (DIR == 1) {
                const float qnan = __int_as_float(0x7fc00000);
                for (int i = tid; 2 * i + par < n_out; i += T) out[2 * i + par] = qnan;
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
            // packed point m of the sub-sequence: (xs[2m], xs[2m+1]) = (x[4m + par], x[4m + 2 + par])
#pragma unroll
            for (int nA = 0; nA < RA; ++nA) {
                const int m = nA * LB + tid;
                v[nA] = make_float2(__ldg(x + 4 * m + par), __ldg(x + 4 * m + 2 + par));
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
            const int m = nA * LB + tid;
            const int j0 = 4 * m + par - a.crop, j1 = j0 + 2;
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

// One thread per k in [0, 16384]: bins k and 32768 - k of the full spectrum.
template <int MODE>
__global__ void __launch_bounds__(256) long_pointwise_kernel(const LongPwArgs a) {
    constexpr int KS = LONG_KS, MS = KS - 1, MF = 2 * MS, KF = MF + 1, NF = 2 * MF;     // MF = 32768 = N/2
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= KS) return;
    const int lu = blockIdx.y;
    const int unit = a.unit0 + lu;
    const int b = unit / a.n_det, d = unit - b * a.n_det;
    float2* se = a.spec + ((size_t)lu * 2) * LONG_KS_STRIDE;
    float2* so = se + LONG_KS_STRIDE;
    float2 A = make_float2(0.f, 0.f), Bq = A;
    if (!a.nofwd) { A = se[k]; Bq = so[k]; }
    const float2 w = twiddle<NF>(k);
    const float2 B = cmul(Bq, w);
    float2 x1 = make_float2(A.x + B.x, A.y + B.y);              // 2 X[k]
    float2 x2 = make_float2(A.x - B.x, -(A.y - B.y));           // 2 X[N/2 - k] = conj(2A - 2B)
    const int k2 = MF - k;
    if (MODE == MODE_HDET) {
        const float2* h = a.h_det + (size_t)unit * KF;
        const float2 h1 = __ldg(h + k), h2 = __ldg(h + k2);
        x1.x = fmaf(a.two_fs, h1.x, x1.x); x1.y = fmaf(a.two_fs, h1.y, x1.y);
        x2.x = fmaf(a.two_fs, h2.x, x2.x); x2.y = fmaf(a.two_fs, h2.y, x2.y);
    } else if (MODE == MODE_FUSED) {
        const WfCoef* c = a.coef + b;
        if (c->valid) {
            const DetResp r = a.resp[unit];
            const float cre = (float)r.fp * c->pol_p;               // C = F+ (1+cos^2 i)/2 - i Fx cos i
            const float cim = -(float)r.fc * c->pol_c;
            const double delta = r.dt * a.inv_tseg;                // turns per bin
            const float2* h = a.h0 + (size_t)b * KF;
            auto inject = [&](int kk, float2& x) {
                if (kk < c->k_lo || kk > c->k_hi) return;
                const float2 hv = __ldg(h + kk);
                double turns = (double)kk * delta;
                turns -= rint(turns);
                float s, co;
                sincospif(-2.0f * (float)turns, &s, &co);           // exp(-2 pi i k dt / T)
                const float2 cp = make_float2(cre * co - cim * s, cre * s + cim * co);
                x.x += hv.x * cp.x - hv.y * cp.y;
                x.y += hv.x * cp.y + hv.y * cp.x;
            };
            inject(k, x1);
            inject(k2, x2);
        }
    }
    const float* filt = a.filt + (size_t)d * a.filt_stride;
    const float f1 = __ldg(filt + k), f2 = __ldg(filt + k2);
    const float2 P = make_float2(x1.x * f1, x1.y * f1);
    const float2 Q = make_float2(x2.x * f2, -x2.y * f2);        // conj(Y[N/2 - k])
    float2 ye = make_float2(P.x + Q.x, P.y + Q.y);
    float2 yo = cmul_conj(make_float2(P.x - Q.x, P.y - Q.y), w);
    if (k == 0 || k == MS) { ye.y = 0.f; yo.y = 0.f; }           // DC / Nyquist of the sub-transforms are real
    se[k] = ye;
    so[k] = yo;
}

static int long_attr() {
    static bool done = false;
    if (done) return AMPLFI_OK;
    cudaError_t e = cudaFuncSetAttribute(long_sub_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)Fft<LONG_LOGM>::SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(long_sub_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)Fft<LONG_LOGM>::SMEM_BYTES);
    if (e != cudaSuccess) { set_error("cudaFuncSetAttribute: %s", cudaGetErrorString(e)); return AMPLFI_ERR_CUDA; }
    done = true;
    return AMPLFI_OK;
}

size_t long_scratch_floats2(int chunk_units) { return (size_t)chunk_units * 2 * LONG_KS_STRIDE; }

int launch_inject_whiten_long(const amplfi_plan* p, const IwArgs& ia, int mode, int units, cudaStream_t st) {
    int rc = long_attr();
    if (rc) return rc;
    using F = Fft<LONG_LOGM>;
    const bool nofwd = ia.noise == nullptr;
    for (int u0 = 0; u0 < units; u0 += p->long_chunk) {
        const int cu = units - u0 < p->long_chunk ? units - u0 : p->long_chunk;
        LongArgs a;
        a.noise = ia.noise; a.offsets = nofwd ? nullptr : ia.offsets; a.strip_len = ia.strip_len; a.spec = p->long_spec;
        a.out = ia.out; a.n_det = ia.n_det; a.unit0 = u0; a.n_full = p->n; a.crop = ia.crop;
        if (!nofwd) { long_sub_kernel<0><<<2 * cu, F::T, F::SMEM_BYTES, st>>>(a); count_launch(); }
        LongPwArgs w;
        w.spec = p->long_spec; w.h_det = ia.h_det; w.h0 = ia.h0; w.coef = ia.coef;
        w.resp = ia.resp; w.filt = ia.filt; w.filt_stride = ia.filt_stride; w.n_det = ia.n_det; w.unit0 = u0;
        w.two_fs = ia.two_fs; w.inv_tseg = 1.0 / p->t_seg; w.nofwd = nofwd ? 1 : 0;
        dim3 grid((LONG_KS + 255) / 256, cu);
        switch (mode) {
            case MODE_NONE: long_pointwise_kernel<MODE_NONE><<<grid, 256, 0, st>>>(w); break;
            case MODE_HDET: long_pointwise_kernel<MODE_HDET><<<grid, 256, 0, st>>>(w); break;
            default: long_pointwise_kernel<MODE_FUSED><<<grid, 256, 0, st>>>(w); break;
        }
        long_sub_kernel<1><<<2 * cu, F::T, F::SMEM_BYTES, st>>>(a);
        count_launch(2);
    }
    return check_launch("inject_whiten_long");
}

}  // namespace amplfi
