// inject_whiten_long.cu -- gather -> FFT -> inject -> whiten -> iFFT for n = 2^18 .. 2^20 (the
// minutes-long segments of binary-neutron-star signals).
// PAPER.md:103, :105 (same step as inject_whiten.cu); "the signal duration can be O(min) ... This makes the
// input arrays larger by an order of magnitude".
//
// Segments of 2^18 .. 2^20 samples (n = 2^16, 2^17 run as thread-block clusters in inject_whiten_v3.cu) exceed what one
// CTA or cluster holds, so the transform is split in four steps around the single-CTA 16384-point complex transform of
// fft_core.cuh (below: "four-step").  Three kernels per chunk of units; a chunk's rows (about 4 n bytes per unit) are sized
// to stay resident in the 126 MB L2, so HBM sees the algorithmic 8 B per sample plus the row copies of h0.
// (Round 1 decimated in time instead -- x[R m + r], strided 4-byte gathers and an O(R) sum per bin -- and was 2 to 3 times
// slower; profiles/r01_configs.md, r02_configs.md.)
#include "amplfi_internal.h"
#include "fft_core.cuh"
#include "waveform.cuh"

namespace amplfi {

constexpr int LONG_LOGM = 14;                       // sub-transform: 16384 complex = 32768 real samples

// exp(-2 pi i num / den) for a power-of-two den <= 2^21: the argument is reduced exactly in integers to [-pi, pi) and
// evaluated with the fast sine/cosine (absolute error ~4e-7, as for the twiddles of the transforms themselves)
__device__ __forceinline__ float2 long_w(long num, int den) {
    int m = (int)(num & (long)(den - 1));
    if (m >= den / 2) m -= den;
    float s, c;
    __sincosf((float)m * (-6.283185307179586f / (float)den), &s, &c);
    return make_float2(c, s);
}

// Four-step transform (decimation in frequency): n = R L with L = 16384, sample index L a + b, bin index c + R e.
//   pass 1  A[c][b] = w_n^(b c) sum_a x[L a + b] w_R^(a c),  c <= R/2        (x real: A[R - c] = conj A[c]); coalesced in b
//   rows    Z[e] = FFT_L(A[c][.]) = X[c + R e] (two-sided); pointwise on the one-sided bin behind it (k = c + R e, or its
//           mirror n - k with everything conjugated); B[c][.] = unnormalised inverse FFT_L; one CTA per (unit, c), in place
//   pass 3  y[L a + b] = Re sum_c w_R^(-a c) D[c][b],  D[c][b] = w_n^(-b c) B[c][b],  D[R - c] = conj D[c]
// Every global access is contiguous in b or e (the first version gathered x[R m + r] at stride R).  The per-bin operands
// of a row (filter, h0) are re-laid out once per call as [c][e] so that the row kernel reads them contiguously too.
constexpr int ROWS_L = 1 << LONG_LOGM;              // 16384 complex points per row

struct LongRowArgs {
    float2* rows;             // [chunk, R/2 + 1, ROWS_L]
    const float* filt_rows;   // [n_det or 1, R/2 + 1, ROWS_L]: filter at the one-sided bin behind (c, e)
    size_t filt_det_stride;   // floats between detectors (0: one filter for all)
    const float2* h0_rows;    // fused: [batch, R/2 + 1, ROWS_L]: 2 fs h0 at the one-sided bin behind (c, e)
    const float2* h_det;      // injected spectra given: [units, n/2 + 1] (read at stride R: rare path)
    const WfCoef* coef;
    const DetResp* resp;
    int n_det, unit0, rdec, nofwd, n_full;
    float two_fs;
    double inv_tseg;
};

template <int MODE>
__global__ void __launch_bounds__(Fft<LONG_LOGM>::T) long_rows_kernel(const LongRowArgs a) {
    using F = Fft<LONG_LOGM>;
    constexpr int L = F::M, RA = F::RA, RC = F::RC, T = F::T, LB = F::LB, RAB = F::RA * F::RB;
    static_assert(F::NA == 1 && F::NB == 1 && RAB == 2 * T, "long_rows_kernel: one butterfly per thread in passes A, B, two in C");
    extern __shared__ float2 sm[];
    const int tid = threadIdx.x;
    const int R = a.rdec, NR = R / 2 + 1;
    const int lu = blockIdx.x / NR, c = blockIdx.x - lu * NR;
    const int unit = a.unit0 + lu;
    const int b = unit / a.n_det, d = unit - b * a.n_det;
    float2* row = a.rows + ((size_t)lu * NR + c) * L;
    const int klow[2] = {tid, tid + T};
    float2 v[2][RC];
    if (!a.nofwd) {
        float2 u[RA];
#pragma unroll
        for (int nA = 0; nA < RA; ++nA) u[nA] = row[nA * LB + tid];
        F::pass_a_fwd(u, tid, sm);
        __syncthreads();
        F::pass_b_fwd(tid, sm);
        __syncthreads();
        F::pass_c_fwd(klow[0], v[0], sm);
        F::pass_c_fwd(klow[1], v[1], sm);
    } else {
#pragma unroll
        for (int i = 0; i < RC; ++i) v[0][i] = v[1][i] = make_float2(0.f, 0.f);
    }
    // ---- a-7, a-8 on the one-sided bin behind two-sided index c + R e (x holds 2 X[k], as in the other kernels) ----
    const float* frow = a.filt_rows + (size_t)d * a.filt_det_stride + (size_t)c * L;
    const int n = a.n_full, mf = n / 2;
    const float2* hrow = nullptr;
    int w_lo = 1, w_hi = 0;
    float cre = 0.f, cim = 0.f;
    double delta = 0.0;
    if (MODE == MODE_HDET) hrow = a.h_det + (size_t)unit * (mf + 1);
    if (MODE == MODE_FUSED) {
        const WfCoef* cf = a.coef + b;
        hrow = a.h0_rows + ((size_t)b * NR + c) * L;
        if (cf->valid) { w_lo = cf->k_lo; w_hi = cf->k_hi; }
        const DetResp r = a.resp[unit];
        cre = (float)r.fp * cf->pol_p;                      // C = F+ (1+cos^2 i)/2 - i Fx cos i
        cim = -(float)r.fc * cf->pol_c;
        delta = r.dt * a.inv_tseg;                          // turns per bin
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
#pragma unroll
        for (int i = 0; i < RC; ++i) {
            const int e = klow[h] + RAB * brev<RC>(i);
            const int k2 = c + R * e;
            const bool direct = k2 <= mf;
            const int k = direct ? k2 : n - k2;
            const float2 z = v[h][i];
            float2 x = make_float2(2.0f * z.x, direct ? 2.0f * z.y : -2.0f * z.y);
            if (MODE == MODE_HDET) {
                const float2 hv = __ldg(hrow + k);
                x.x = fmaf(a.two_fs, hv.x, x.x);
                x.y = fmaf(a.two_fs, hv.y, x.y);
            } else if (MODE == MODE_FUSED) {
                if (k >= w_lo && k <= w_hi) {
                    const float2 hv = __ldg(hrow + e);
                    double turns = (double)k * delta;
                    turns -= rint(turns);
                    float sn, co;
                    __sincosf((float)turns * -6.283185307179586f, &sn, &co);   // exp(-2 pi i k dt / T)
                    const float2 cp = make_float2(cre * co - cim * sn, cre * sn + cim * co);
                    x.x += hv.x * cp.x - hv.y * cp.y;
                    x.y += hv.x * cp.y + hv.y * cp.x;
                }
            }
            const float f = __ldg(frow + e);
            float2 y = make_float2(x.x * f, x.y * f);
            if (k == 0 || k == mf) y.y = 0.f;                   // DC / Nyquist of a real sequence
            v[h][i] = make_float2(y.x, direct ? y.y : -y.y);
        }
    }
    // ---- inverse row transform (unnormalised: the filter carries the 1/(2n)), in place ----
    F::pass_c_inv(klow[0], v[0], sm);
    F::pass_c_inv(klow[1], v[1], sm);
    __syncthreads();
    F::pass_b_inv(tid, sm);
    __syncthreads();
    {
        float2 u[RA];
        F::pass_a_inv(u, tid, sm);
#pragma unroll
        for (int nA = 0; nA < RA; ++nA) row[nA * LB + tid] = u[nA];
    }
}

struct LongEdgeArgs {
    const float* noise;
    const long* offsets;
    long strip_len;
    float2* rows;
    float* out;
    int n_det, unit0, n_full, crop;
};

// cos / sin of 2 pi i / 64, i < 32 (the one stage of the 64-point register transform that fft_core.cuh does not cover)
__device__ constexpr float kCos64[32] = {1.000000000e+00f, 9.951847267e-01f, 9.807852804e-01f, 9.569403357e-01f, 9.238795325e-01f, 8.819212643e-01f, 8.314696123e-01f, 7.730104534e-01f, 7.071067812e-01f, 6.343932842e-01f, 5.555702330e-01f, 4.713967368e-01f, 3.826834324e-01f, 2.902846773e-01f, 1.950903220e-01f, 9.801714033e-02f, 0.000000000e+00f, -9.801714033e-02f, -1.950903220e-01f, -2.902846773e-01f, -3.826834324e-01f, -4.713967368e-01f, -5.555702330e-01f, -6.343932842e-01f, -7.071067812e-01f, -7.730104534e-01f, -8.314696123e-01f, -8.819212643e-01f, -9.238795325e-01f, -9.569403357e-01f, -9.807852804e-01f, -9.951847267e-01f};
__device__ constexpr float kSin64[32] = {0.000000000e+00f, 9.801714033e-02f, 1.950903220e-01f, 2.902846773e-01f, 3.826834324e-01f, 4.713967368e-01f, 5.555702330e-01f, 6.343932842e-01f, 7.071067812e-01f, 7.730104534e-01f, 8.314696123e-01f, 8.819212643e-01f, 9.238795325e-01f, 9.569403357e-01f, 9.807852804e-01f, 9.951847267e-01f, 1.000000000e+00f, 9.951847267e-01f, 9.807852804e-01f, 9.569403357e-01f, 9.238795325e-01f, 8.819212643e-01f, 8.314696123e-01f, 7.730104534e-01f, 7.071067812e-01f, 6.343932842e-01f, 5.555702330e-01f, 4.713967368e-01f, 3.826834324e-01f, 2.902846773e-01f, 1.950903220e-01f, 9.801714033e-02f};

// R-point transforms in registers for R = 16, 32 (fft_core.cuh) and 64 (one radix-2 stage around two 32-point ones):
// forward: natural-order input, output c left in v[edge_pos<R>(c)];  inverse (unnormalised): input c taken from there,
// natural-order output
template <int R>
__host__ __device__ constexpr int edge_pos(int c) { return R <= 32 ? brev<(R <= 32 ? R : 32)>(c) : (c & 1) * 32 + brev<32>(c >> 1); }
template <int R>
__device__ __forceinline__ void edge_fft_fwd(float2 (&v)[R]) {
    if constexpr (R <= 32) {
        fft_dif_fwd<R>(v);
    } else {
        float2 lo[32], hi[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            lo[i] = cadd(v[i], v[i + 32]);
            hi[i] = cmul(csub(v[i], v[i + 32]), make_float2(kCos64[i], -kSin64[i]));      // w_64^i
        }
        fft_dif_fwd<32>(lo);                                    // even c
        fft_dif_fwd<32>(hi);                                    // odd c
#pragma unroll
        for (int i = 0; i < 32; ++i) { v[i] = lo[i]; v[i + 32] = hi[i]; }
    }
}
template <int R>
__device__ __forceinline__ void edge_fft_inv(float2 (&v)[R]) {
    if constexpr (R <= 32) {
        fft_dit_inv<R>(v);
    } else {
        float2 lo[32], hi[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) { lo[i] = v[i]; hi[i] = v[i + 32]; }
        fft_dit_inv<32>(lo);
        fft_dit_inv<32>(hi);
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            const float2 t = cmul_conj(hi[i], make_float2(kCos64[i], -kSin64[i]));
            v[i] = cadd(lo[i], t);
            v[i + 32] = csub(lo[i], t);
        }
    }
}

// pass 1 (DIR = 0) and pass 3 (DIR = 1): one thread per b, an R-point transform in registers across the R blocks of L
template <int R, int DIR>
__global__ void __launch_bounds__(256) long_edge_kernel(const LongEdgeArgs a) {
    constexpr int L = ROWS_L, NR = R / 2 + 1;
    const int b = blockIdx.x * blockDim.x + threadIdx.x;       // < L (L is a multiple of the block size)
    const int lu = blockIdx.y, unit = a.unit0 + lu, d = unit % a.n_det;
    const int n = a.n_full;
    float2* rows = a.rows + (size_t)lu * NR * L + b;
    bool bad = false;
    const float* x = nullptr;
    if (a.noise != nullptr) {
        if (a.offsets != nullptr) {
            const long off = a.offsets[unit];
            bad = off < 0 || off + n > a.strip_len;             // never read out of bounds: the row is poisoned instead
            x = a.noise + (size_t)d * a.strip_len + (bad ? 0 : off);
        } else {
            x = a.noise + (size_t)unit * n;
        }
    }
    const float2 w1 = long_w((long)b, n);                       // w_n^b
    float2 v[R];
    if (DIR == 0) {
        if (bad) return;                                        // pass 3 writes the NaN row
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = make_float2(__ldg(x + (size_t)q * L + b), 0.f);
        edge_fft_fwd<R>(v);                                     // sum_a x[L a + b] w_R^(a c) in v[edge_pos<R>(c)]
        float2 wr = make_float2(1.f, 0.f);
#pragma unroll
        for (int c = 0; c < NR; ++c) {
            if ((c & 7) == 0 && c > 0) wr = long_w((long)c * b, n);
            rows[(size_t)c * L] = cmul(v[edge_pos<R>(c)], wr);
            wr = cmul(wr, w1);
        }
    } else {
        const int n_out = n - 2 * a.crop;
        float* out = a.out + (size_t)unit * n_out;
        if (bad) {
            const float qnan = __int_as_float(0x7fc00000);
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const int i = q * L + b - a.crop;
                if (i >= 0 && i < n_out) out[i] = qnan;
            }
            return;
        }
        float2 wr = make_float2(1.f, 0.f);
#pragma unroll
        for (int c = 0; c < NR; ++c) {
            if ((c & 7) == 0 && c > 0) wr = long_w((long)c * b, n);
            const float2 dv = cmul_conj(rows[(size_t)c * L], wr);      // D[c][b] = w_n^(-b c) B[c][b]
            v[edge_pos<R>(c)] = dv;
            if (c > 0 && c < R / 2) v[edge_pos<R>(R - c)] = make_float2(dv.x, -dv.y);
            wr = cmul(wr, w1);
        }
        edge_fft_inv<R>(v);                                     // natural order: a
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const int i = q * L + b - a.crop;
            if (i >= 0 && i < n_out) __stcs(out + i, v[q].x);
        }
    }
}

// rows[c][e] = src[one-sided bin behind two-sided index c + R e]  (TT = float: filter; float2: h0), c <= R/2.
// coef != nullptr (h0): item = sample, and only the bins within 64 of the sample's band are copied (the row kernel reads
// h0 inside the band only; the linear h0 row is written only there).
template <class TT>
__global__ void __launch_bounds__(256) long_relayout_kernel(const TT* __restrict__ src, size_t src_stride, TT* __restrict__ dst,
                                                            const WfCoef* __restrict__ coef, int rdec, int n) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;       // < ROWS_L
    const int c = blockIdx.y, item = blockIdx.z;
    const int k2 = c + rdec * e;
    const int k = k2 <= n / 2 ? k2 : n - k2;
    if (coef != nullptr) {
        const WfCoef& cf = coef[item];
        if (!cf.valid || k < cf.k_lo - 64 || k > cf.k_hi + 64) return;
    }
    dst[((size_t)item * (rdec / 2 + 1) + c) * ROWS_L + e] = src[(size_t)item * src_stride + k];
}

size_t long_scratch_floats2(int chunk_units, int rdec) { return (size_t)chunk_units * (rdec / 2 + 1) * ROWS_L; }
size_t long_row_elems(int rdec) { return (size_t)(rdec / 2 + 1) * ROWS_L; }

template <int R>
static void launch_long_edges(const LongEdgeArgs& e, int dir, int cu, cudaStream_t st) {
    dim3 grid(ROWS_L / 256, cu);
    if (dir == 0) long_edge_kernel<R, 0><<<grid, 256, 0, st>>>(e);
    else long_edge_kernel<R, 1><<<grid, 256, 0, st>>>(e);
    count_launch();
}

int launch_inject_whiten_long(const amplfi_plan* p, const IwArgs& ia, int mode, int units, cudaStream_t st) {
    using F = Fft<LONG_LOGM>;
    static std::atomic<unsigned> done0{0}, done1{0}, done2{0};
    int rc = ensure_dynamic_smem(long_rows_kernel<MODE_NONE>, (int)F::SMEM_BYTES, done0);
    if (!rc) rc = ensure_dynamic_smem(long_rows_kernel<MODE_HDET>, (int)F::SMEM_BYTES, done1);
    if (!rc) rc = ensure_dynamic_smem(long_rows_kernel<MODE_FUSED>, (int)F::SMEM_BYTES, done2);
    if (rc) return rc;
    const bool nofwd = ia.noise == nullptr;
    const int R = p->n / ROWS_L, NR = R / 2 + 1;
    if (R != 16 && R != 32 && R != 64) { set_error("inject_whiten_long: n = %d not supported", p->n); return AMPLFI_ERR_UNSUPPORTED_SIZE; }
    // operands of the rows, once per call: the filter of every detector and, on the fused path, h0 of every sample
    const int n_filt = ia.filt_stride ? ia.n_det : 1;
    {
        dim3 g(ROWS_L / 256, NR, n_filt);
        long_relayout_kernel<float><<<g, 256, 0, st>>>(ia.filt, (size_t)ia.filt_stride, p->long_filt_rows, nullptr, R, p->n);
        count_launch();
    }
    if (mode == MODE_FUSED) {
        const int batch = units / ia.n_det;
        dim3 g(ROWS_L / 256, NR, batch);
        long_relayout_kernel<float2><<<g, 256, 0, st>>>(ia.h0, (size_t)(p->n / 2 + 1), p->long_h0_rows, ia.coef, R, p->n);
        count_launch();
    }
    for (int u0 = 0; u0 < units; u0 += p->long_chunk) {
        const int cu = units - u0 < p->long_chunk ? units - u0 : p->long_chunk;
        LongEdgeArgs e;
        e.noise = ia.noise; e.offsets = nofwd ? nullptr : ia.offsets; e.strip_len = ia.strip_len; e.rows = p->long_spec;
        e.out = ia.out; e.n_det = ia.n_det; e.unit0 = u0; e.n_full = p->n; e.crop = ia.crop;
        if (!nofwd) {
            if (R == 16) launch_long_edges<16>(e, 0, cu, st);
            else if (R == 32) launch_long_edges<32>(e, 0, cu, st);
            else launch_long_edges<64>(e, 0, cu, st);
        }
        LongRowArgs w;
        w.rows = p->long_spec; w.filt_rows = p->long_filt_rows; w.filt_det_stride = ia.filt_stride ? long_row_elems(R) : 0;
        w.h0_rows = p->long_h0_rows; w.h_det = ia.h_det; w.coef = ia.coef; w.resp = ia.resp;
        w.n_det = ia.n_det; w.unit0 = u0; w.rdec = R; w.nofwd = nofwd ? 1 : 0; w.n_full = p->n;
        w.two_fs = ia.two_fs; w.inv_tseg = 1.0 / p->t_seg;
        switch (mode) {
            case MODE_NONE: long_rows_kernel<MODE_NONE><<<cu * NR, F::T, F::SMEM_BYTES, st>>>(w); break;
            case MODE_HDET: long_rows_kernel<MODE_HDET><<<cu * NR, F::T, F::SMEM_BYTES, st>>>(w); break;
            default: long_rows_kernel<MODE_FUSED><<<cu * NR, F::T, F::SMEM_BYTES, st>>>(w); break;
        }
        count_launch();
        if (R == 16) launch_long_edges<16>(e, 1, cu, st);
        else if (R == 32) launch_long_edges<32>(e, 1, cu, st);
        else launch_long_edges<64>(e, 1, cu, st);
    }
    return check_launch("inject_whiten_long");
}

}  // namespace amplfi
