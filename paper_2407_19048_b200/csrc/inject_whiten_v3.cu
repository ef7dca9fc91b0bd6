// inject_whiten_v3.cu -- fused gather -> FFT -> inject -> whiten -> iFFT, third generation (n = 4096 ... 131072; all five configs).
// PAPER.md:103 (background chunks sliced from the GPU-resident strip), PAPER.md:105 (inject, whiten with the estimated PSD).
//
// M = 8192 complex points = 32 * 16 * 16: THREE passes per direction (two shared-memory exchanges instead of three),
// 256 threads x 32 points, two CTAs per SM.  Every pass is a radix-2 decimation-in-time network whose butterflies carry
// the inter-pass twiddle in cosine-tangent form (fft_tan.cuh: 6 FMA per butterfly, no separate twiddle multiplication).
//
// Index algebra.  n = 256 n1 + 16 n2 + n3,  k = k1 + 32 k2 + 512 k3  (n1, k1 < 32; n2, n3, k2, k3 < 16);
//   n k / M = n1 k1/32 + n2 k1/512 + n2 k2/16 + n3 (k1 + 32 k2)/8192 + n3 k3/16   (mod 1)
//   FA  thread j = 16 n2 + n3:     A[k1; j]      = sum_n1 z[256 n1 + j] w32^(n1 k1)            operands from global memory;
//                                  scalar radix-2 stage (n1, n1 + 16), then lanes (even k1 | odd k1) run one packed DFT16
//   FB  thread (kap, n3):          B[k1, k2; n3] = sum_n2 A[k1; n2, n3] w512^(n2 k1) w16^(n2 k2)   lanes k1 = 2 kap | 2 kap + 1
//   FC  thread t: klow = k1 + 32 k2 = t (lane A) and 512 - t (lane B; t = 0: 256):
//                                  Z[klow + 512 k3] = sum_n3 B[klow; n3] w8192^(n3 klow) w16^(n3 k3)
//       bins k and M - k meet in one thread (A[k3] <-> B[15 - k3]): split / inject / whiten / merge in registers
//   I1  same threads:              C[klow; n3]   = sum_k3 Y[klow + 512 k3] w16^(-n3 k3)
//   I2  thread (kap, n3):          D[k1; n2, n3] = sum_k2 C[k1, k2; n3] w256^(-n3 k2) w16^(-n2 k2)
//   I3  thread j:                  y[256 n1 + j] = sum_k1 D[k1; j] w8192^(-k1 j) w32^(-n1 k1)   packed DFT16 on the lanes
//                                  (even k1 | odd k1), scalar last radix-2 stage, natural-order float2 stores
// Twiddles: FA / I1 exact constants; FB / I2 from two 2 KB tables (fp64-computed); FC / I3 depend on the whole thread index
// and are evaluated on the fly (fast sincos + reciprocal; every angle lies in [-pi, 0], no range reduction).
//
// Shared memory: two float planes, element (d2, n3, k1) at d2*544 + n3*34 + k1 (d2 = n2 or k2).  The row padding 32 -> 34
// makes the 64-bit (lane A, lane B) accesses of FA/FB/I2/I3 and the 32-bit accesses of FC/I1 bank-conflict free with
// immediate offsets only (no swizzle arithmetic).  Every pass works in place: 4 barriers per segment.
#include <cooperative_groups.h>

#include "amplfi_internal.h"
#include "fft_tan.cuh"
#include "spec_layout.cuh"
#include "waveform.cuh"

namespace amplfi {
namespace v3 {

using namespace tn;

// Geometry of a segment length: M = 2^LOGM = 32 * RB * 16 complex points, RB = 16 / 8 / 4 for n = 16384 / 8192 / 4096
// (the paper's own 4 s at 2048 Hz is n = 8192); T = M/32 threads (256 / 128 / 64), 2 / 4 / 8 CTAs per SM.
// Pass FB / I2 is then a radix RB, of which every thread takes 16/RB.
// n = 32768 (LOGM = 14): M = 32 * (4 * 8) * 16, the middle pass split in two (FB1 radix 4 over n2a, FB2 radix 8 over
// n2b; a third exchange), 512 threads, one CTA per SM.
// n = 65536 (LOGM = 15): M = 32 * (8 * 8) * 16 does not fit one SM's shared memory (256 KB + padding), so a CLUSTER OF TWO
// CTAs of 512 threads holds it: CTA r owns the elements with n3 in [8r, 8r + 8), i.e. element (d2, n3, k1) sits in CTA
// n3 >> 3 at d2 * 272 + (n3 & 7) * 34 + k1.  FA, FB1, FB2 and I2b, I2a, I3 then touch their own CTA only; FC reads half
// of its operands from the peer through distributed shared memory and I1 writes half of its results there: one remote
// exchange per direction, bracketed by the two cluster barriers.
// n = 131072 (LOGM = 16): the same with M = 32 * (8 * 16) * 16 in a cluster of FOUR CTAs, four rows n3 each (element
// (d2, n3, k1) in CTA n3 >> 2 at d2 * 136 + (n3 & 3) * 34 + k1); three quarters of every FC column are remote.
template <int LOGM>
struct Geo {
    static constexpr int M = 1 << LOGM, N = 2 * M, K = M + 1;
    static constexpr int T = M / 32;                  // threads per segment
    static constexpr int CL = LOGM >= 15 ? 1 << (LOGM - 14) : 1;     // CTAs per segment (cluster size: 2, 4)
    static constexpr int NR = 16 / CL;                // rows n3 of a column held by one CTA
    static constexpr int RB2 = LOGM == 16 ? 16 : 8;   // LOGM >= 14: radix of the second half of the middle pass
    static constexpr int TC = T / CL;                 // threads per CTA
    static constexpr int KL = M / 16;                 // span of klow = k1 + 32 k2
    static constexpr int RB = LOGM <= 13 ? M / 512 : (LOGM == 14 ? 4 : 8);   // radix of the middle pass (LOGM >= 14: of its first half)
    static constexpr int NB = 16 / RB;                // middle-pass butterflies per thread
    static constexpr int PLANE = (M / 512) * 544 / CL;    // floats per plane and CTA
    static constexpr int SMEM_BYTES = 2 * PLANE * (int)sizeof(float);
    static constexpr int CTAS = TC >= 512 ? 1 : 512 / TC; // per SM (registers: 128 per thread)
};
constexpr int ROW = 34, BLK = 16 * ROW;               // 34, 544 floats

// FB: per-lane twiddles of W = w_(32 RB)^k1, k1 = 2 kap (lane A), 2 kap + 1 (lane B): (cA, cB, tauA, tauB)
// I2: shared twiddles of W = w_(16 RB)^n3 (used conjugated): (c, tau)
// rows in the layout fft_tan.cuh gives each radix; one set per segment length [LOGM - 11].
// LOGM = 14: fb1 W = w_128^k1 [kap], fb2 W = w_1024^(k1 + 32 k2a) [4 kap + k2a], i2b W = w_128^n3 [n3],
//            i2a W = w_512^(n3 + 16 n2b) [16 n2b + n3].
struct Tables {
    float4 fb[3][16][8];
    float2 i2[3][16][8];
    float4 fb1_14[16][2], fb2_14[64][4];
    float2 i2b_14[16][4], i2a_14[128][2];
    // LOGM = 15: fb1 W = w_256^k1 [kap], fb2 W = w_2048^(k1 + 32 k2a) [8 kap + k2a], i2b W = w_128^n3 [n3],
    //            i2a W = w_1024^(n3 + 16 n2b) [16 n2b + n3]; radix-8 rows (W^4, W^2, W, W w8)
    // (n = 131072, [1]: fb2 and i2b are radix-16 rows, i2a has 256 rows 16 n2b + n3)
    float4 fb1_c[2][16][4], fb2_c[2][128][8];
    float2 i2b_c[2][16][8], i2a_c[2][256][4];
};
static __device__ Tables g_tab;

__device__ __forceinline__ C2 lds2(const float* re, const float* im, int o) {
    return C2{*reinterpret_cast<const u64*>(re + o), *reinterpret_cast<const u64*>(im + o)};
}
__device__ __forceinline__ void sts2(float* re, float* im, int o, C2 v) {
    *reinterpret_cast<u64*>(re + o) = v.r;
    *reinterpret_cast<u64*>(im + o) = v.i;
}

// the eight twiddles of a radix-16 pass with W = w_M^x (fft_tan.cuh: W^8, W^4, W^2, W^2 w8, W w16^q), theta = -(2 pi / M) e;
// every exponent e stays at or below M/2 for the callers' x, so theta lies in [-pi, 0] (no range reduction)
template <int M>
__device__ __forceinline__ void pass_twiddles(float x, Tw1 (&tw)[8]) {
    constexpr float u = -6.283185307179586f / (float)M;
    tw[0] = tan_twiddle(x * (8.0f * u));
    tw[1] = tan_twiddle(x * (4.0f * u));
    tw[2] = tan_twiddle(x * (2.0f * u));
    tw[3] = tan_twiddle(fmaf(x, 2.0f * u, (float)(M / 8) * u));
#pragma unroll
    for (int q = 0; q < 4; ++q) tw[4 + q] = tan_twiddle(fmaf(x, u, (float)(M / 16 * q) * u));
}

// VIEWS = 2 (fused mode, n <= 16384): the two data views d, d' of one background segment from ONE forward
// transform.  After pass FC every thread parks its 16 packed spectrum values in the second view's own output row (16 bytes x
// 16 x T = exactly one row, L2-resident), finishes the first view, reads them back and runs the pointwise stage with the
// arrival time later by t_shift[b] and the inverse transform into that row.
template <int LOGM, int MODE, bool FWD, int VIEWS = 1>
__global__ void __launch_bounds__(Geo<LOGM>::TC, Geo<LOGM>::CTAS) inject_whiten3_kernel(const IwArgs a, int units) {
    using G = Geo<LOGM>;
    constexpr int M = G::M, N = G::N, K = G::K, T = G::T, TC = G::TC, KL = G::KL, RB = G::RB, NB = G::NB, PLANE = G::PLANE;
    namespace cg = cooperative_groups;
    extern __shared__ float smem3[];
    float* re = smem3;
    float* im = smem3 + PLANE;
    __shared__ float4 sp[8];          // (S[2w].re, S[2w+1].re, S[2w].im, S[2w+1].im), S[u] = exp(-2 pi i 512 u dt/T)
    __shared__ float2 s_em;           // exp(-2 pi i M dt/T)
    __shared__ float2 sc[32];         // the two self-paired butterflies of thread 0
    __shared__ float4 sx[17][2];      // their operands, prepared by lanes 0..16 of warp 0 long before they are needed
    __shared__ float4 sraw[17];       // VIEWS = 2: the h0 values those operands are built from, kept for the second view
    // LOGM = 15: blocks 2u and 2u + 1 form the cluster of unit u; t is the thread's index within the segment
    constexpr int CL = G::CL, NR = G::NR, RB2 = G::RB2, BLKC = NR * ROW;      // cluster geometry (CL = 1: unused)
    const int rank = CL > 1 ? (int)(blockIdx.x & (CL - 1)) : 0;
    const int unit = CL > 1 ? (int)(blockIdx.x / CL) : (int)blockIdx.x, tid = threadIdx.x;
    const int t = rank * TC + tid;
    const int b = unit / a.n_det, d = unit - b * a.n_det;
    // the planes of CTA c of the cluster (generic addresses; mapped where they are used, so that no pointer stays live)
    auto peer_re = [&](int c) { return cg::this_cluster().map_shared_rank(re, c); };
    auto peer_im = [&](int c) { return cg::this_cluster().map_shared_rank(im, c); };
    // run `body` with the CTA's rank as a compile-time constant (row ownership then selects plain shared-memory accesses)
    auto with_rank = [&](auto body) {
        if constexpr (CL == 2) {
            if (rank == 0) body(std::integral_constant<int, 0>{}); else body(std::integral_constant<int, 1>{});
        } else if constexpr (CL == 4) {
            switch (rank) {
                case 0: body(std::integral_constant<int, 0>{}); break;
                case 1: body(std::integral_constant<int, 1>{}); break;
                case 2: body(std::integral_constant<int, 2>{}); break;
                default: body(std::integral_constant<int, 3>{}); break;
            }
        }
    };

    // ---- a-5 gather ----
    const float* x = nullptr;
    const int n_out = N - 2 * a.crop;
    float* out = a.out + (size_t)unit * n_out;
    if (!FWD) {
    } else if (a.offsets != nullptr) {
        const long off = a.offsets[unit];
        if (off < 0 || off + N > a.strip_len) {            // never read out of bounds: poison the row instead
            const float qnan = __int_as_float(0x7fc00000);
            for (int i = t; i < n_out; i += T) out[i] = qnan;
            if (VIEWS == 2) {
                float* o2 = a.out2 + (size_t)unit * n_out;
                for (int i = t; i < n_out; i += T) o2[i] = qnan;
            }
            return;
        }
        x = a.noise + (size_t)d * a.strip_len + off;
    } else {
        x = a.noise + (size_t)unit * N;
    }
    // L2 prefetch of the segment a CTA two waves later will gather (one bulk instruction for the whole 64 KB)
    if (t == 0 && FWD) {
        const int nu = unit + a.prefetch_ahead;
        if (nu < units) {
            const float* nx;
            bool ok = true;
            if (a.offsets != nullptr) {
                const long noff = a.offsets[nu];
                ok = noff >= 0 && noff + N <= a.strip_len;
                nx = a.noise + (size_t)(nu % a.n_det) * a.strip_len + noff;
            } else {
                nx = a.noise + (size_t)nu * N;
            }
            const size_t p0 = (reinterpret_cast<size_t>(nx) + 15) & ~(size_t)15;      // inside the segment
            if (ok) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p0), "r"(N * 4 - 16) : "memory");
        }
    }

    // FA / I3: point j = 16 n2 + n3 (one CTA: j = tid; cluster: the CTA's NR values of n3)
    const int n3l = CL > 1 ? tid & (NR - 1) : tid & 15;      // row within the CTA
    const int n2 = CL > 1 ? tid / NR : tid >> 4, n3 = CL > 1 ? NR * rank + n3l : n3l;
    const int j = 16 * n2 + n3;
    const int oj = CL > 1 ? n2 * BLKC + n3l * ROW : n2 * BLK + n3 * ROW;     // element (n2, n3, k1 = 0)
    // FB / I2: butterfly i of this thread is (kap, n3) = ((tid + T i) >> 4, tid & 15): element (d2 = 0, n3, k1 = 2 kap)
    auto ob_of = [&](int i) { return n3 * ROW + 2 * ((tid + T * i) >> 4); };

    // ---- FA: radix 32 over n1, operands from global memory ----
    if (FWD) {
        float2 z[32];
        if ((reinterpret_cast<size_t>(x) & 7) == 0) {
            const float2* x2 = reinterpret_cast<const float2*>(x) + j;
#pragma unroll
            for (int n1 = 0; n1 < 32; ++n1) z[n1] = __ldcs(x2 + n1 * T);
        } else {
#pragma unroll
            for (int n1 = 0; n1 < 32; ++n1) {
                const int m = n1 * T + j;
                z[n1] = make_float2(__ldg(x + 2 * m), __ldg(x + 2 * m + 1));
            }
        }
        C2 v[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const float2 s = amplfi::cadd(z[r], z[r + 16]);
            float2 df = amplfi::csub(z[r], z[r + 16]);
            switch (r) {      // df *= w32^r
                case 0: break;
                case 1: df = mul_w32<1, false>(df); break;
                case 2: df = mul_w32<2, false>(df); break;
                case 3: df = mul_w32<3, false>(df); break;
                case 4: df = mul_w32<4, false>(df); break;
                case 5: df = mul_w32<5, false>(df); break;
                case 6: df = mul_w32<6, false>(df); break;
                case 7: df = mul_w32<7, false>(df); break;
                case 8: df = mul_w32<8, false>(df); break;
                case 9: df = mul_w32<9, false>(df); break;
                case 10: df = mul_w32<10, false>(df); break;
                case 11: df = mul_w32<11, false>(df); break;
                case 12: df = mul_w32<12, false>(df); break;
                case 13: df = mul_w32<13, false>(df); break;
                case 14: df = mul_w32<14, false>(df); break;
                default: df = mul_w32<15, false>(df); break;
            }
            v[brev<16>(r)] = C2{pack(s.x, df.x), pack(s.y, df.y)};
        }
        dit16_const<false>(v);
#pragma unroll
        for (int kap = 0; kap < 16; ++kap) sts2(re, im, oj + 2 * kap, v[kap]);
    }
    // ---- per-unit constants of the pointwise stage ----
    const float* hsrc = nullptr;                             // HDET: complex spectrum as floats, re at 2k, im at 2k + 1
    int w_lo = 0x40000000, w_hi = -1;                        // empty band
    float cre = 0.f, cim = 0.f;
    double delta = 0.0;
    if (MODE == MODE_HDET) hsrc = reinterpret_cast<const float*>(a.h_det + (size_t)unit * K);
    if (MODE == MODE_FUSED) {
        const WfCoef* c = a.coef + b;
        hsrc = reinterpret_cast<const float*>(a.h0) + (size_t)b * (2 * M);              // slot layout
        if (c->valid) { w_lo = c->k_lo; w_hi = c->k_hi; }       // an empty band is stored as (2^30, -1) by prepare_kernel
        const DetResp r = a.resp[unit];
        cre = (float)r.fp * c->pol_p;                       // C = F+ (1+cos^2 i)/2 - i Fx cos i
        cim = -(float)r.fc * c->pol_c;
        delta = r.dt * (double)a.inv_tseg;                   // turns per bin
    }
    auto unit_phase = [&](int k) {                           // exp(-2 pi i k delta)
        float turns;
        if (a.phase64) { const double xx = (double)k * delta; turns = (float)(xx - rint(xx)); }
        else { turns = (float)k * (float)delta; turns -= rintf(turns); }
        float s, co;
        __sincosf(turns * -6.283185307179586f, &s, &co);
        return make_float2(co, s);
    };
    auto view_constants = [&]() {                            // the S table and e(M) of the current arrival time
        if (MODE == MODE_FUSED && tid <= 16) {
            if (tid < 16) {
                const float2 e = unit_phase(KL * tid);
                float* spf = reinterpret_cast<float*>(sp);
                spf[(tid >> 1) * 4 + (tid & 1)] = e.x;
                spf[(tid >> 1) * 4 + 2 + (tid & 1)] = e.y;
            } else {
                s_em = unit_phase(M);
            }
        }
    };
    view_constants();

    // Operands of the pointwise stage in the slot layout (spec_layout.cuh): pulled into L1 now, a whole pass ahead of
    // their use, so that the 16-byte requests of the pointwise stage find them there instead of waiting on L2.
    unsigned need = 0;                                       // bit w: first h0 slots of unit w needed, bit 8 + w: second
    if (MODE == MODE_FUSED) {
        const int l = t & 31;
        need = __ballot_sync(0xffffffffu, l < 16 && slot::window_needed(KL, l >> 3, l & 7, t >> 5, w_lo, w_hi));
    }
    const float4* fsl = reinterpret_cast<const float4*>(a.filt_slots) + (a.filt_stride ? d * (M / 4) : 0) + t;
    const float4* hsl = reinterpret_cast<const float4*>(a.h0) + (size_t)b * (M / 2) + t;
    if ((t & 7) == 0) {                                      // one request per 128-byte line
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            asm volatile("prefetch.global.L1 [%0];" ::"l"(fsl + w * T));
            if (MODE == MODE_FUSED) {
                if (need & (1u << w)) asm volatile("prefetch.global.L1 [%0];" ::"l"(hsl + w * T));
                if (need & (256u << w)) asm volatile("prefetch.global.L1 [%0];" ::"l"(hsl + (8 + w) * T));
            }
        }
    }

    // Operands of the self-paired butterflies klow = 0 and 256 (thread 0 holds them; lanes 0..16 of warp 0 process their
    // 17 bin pairs after the unit loop): lane 0: Z[0] (DC and Nyquist); lanes 1..7: k = 512 l; lane 8: k = M/2;
    // lanes 9..16: k = 256 + 512 (l - 9).  Requested here, turned into (filter values, injected terms, split twiddle)
    // after pass FB and parked in shared memory, so that nothing in that late section waits on memory.
    // (prepared by lanes 0..16 of the LAST warp, so that warp 0 does not carry all the extra work of these butterflies)
    const int sl = rank == 0 ? tid - (TC - 32) : -1;         // task index of this thread, valid if 0 <= sl <= 16 (CTA 0 holds thread 0)
    const int sk = sl <= 0 ? 0 : (sl <= 8 ? KL * sl : KL / 2 + KL * (sl - 9));
    float sfa = 0.f, sfb = 0.f;
    float2 sha = make_float2(0.f, 0.f), shb = make_float2(0.f, 0.f);
    bool sin_a = false, sin_b = false;
    auto special_loads = [&]() {
    if (sl >= 0 && sl <= 16) {
        const float* filt = a.filt + (size_t)d * a.filt_stride;
        sfa = __ldg(filt + sk);
        sfb = __ldg(filt + M - sk);
        if (MODE == MODE_HDET) {
            sha = make_float2(__ldg(hsrc + 2 * sk), __ldg(hsrc + 2 * sk + 1));
            shb = make_float2(__ldg(hsrc + 2 * (M - sk)), __ldg(hsrc + 2 * (M - sk) + 1));
        } else if (MODE == MODE_FUSED && sl != 0) {
            sin_a = sk >= w_lo && sk <= w_hi;
            sin_b = M - sk >= w_lo && M - sk <= w_hi;
            if (sin_a) { const float* hp = hsrc + slot::h0_index(KL, sk); sha = make_float2(__ldg(hp), __ldg(hp + 2)); }
            if (sin_b) { const float* hp = hsrc + slot::h0_index(KL, M - sk); shb = make_float2(__ldg(hp), __ldg(hp + 2)); }
        }
    }
    };
    special_loads();

    // the factor conj(w32^n3) of the self-paired column klow = KL/2 (lane B of thread 0 in FC, whose twiddles are those of
    // klow = 0, i.e. 1): one complex product in the 16 threads that produce that column
    auto column_factor = [&](C2& v) {
        float ar_, br_, ai_, bi_;
        unpack(v.r, ar_, br_);
        unpack(v.i, ai_, bi_);
        const float co = kCos32[n3], si = kSin32[n3];
        v = C2{pack(ar_ * co - ai_ * si, br_), pack(ar_ * si + ai_ * co, bi_)};
    };
    if constexpr (LOGM <= 13) {
    // ---- FB: radix RB over n2 (NB butterflies per thread) ----
    if (FWD) {
        Tw2 tw[NB][8];
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
            for (int e = 0; e < (RB == 16 ? 8 : (RB == 8 ? 4 : 2)); ++e) {
                const float4 f = __ldg(&g_tab.fb[LOGM - 11][(tid + T * i) >> 4][e]);
                tw[i][e] = Tw2{pack(f.x, f.y), pack(f.z, f.w)};
            }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int ob = ob_of(i);
            C2 v[RB];
#pragma unroll
            for (int r = 0; r < RB; ++r) v[brev<RB>(r)] = lds2(re, im, ob + r * BLK);
            dit_r<RB, false, Tw2, true>(v, tw[i]);           // k2 >= RB/2 (the klow >= KL/2 read by lane B of FC) stored conjugated
            if (((tid + T * i) >> 4) == 0) column_factor(v[RB / 2]);        // column KL/2: k1 = 0, k2 = RB/2
#pragma unroll
            for (int k2 = 0; k2 < RB; ++k2) sts2(re, im, ob + k2 * BLK, v[k2]);
        }
    }
    } else if constexpr (CL > 1) {
    // ---- clusters (n = 65536, 131072): FB1 radix 8 over n2a, FB2 radix RB2 = 8 / 16 over n2b, both inside the CTA ----
    // element (d2a, d2b, n3l, k1) at (RB2 d2a + d2b) * BLKC + n3l * ROW + k1.  The lane bits above n3l are given to indices that
    // move the address by 8 / 16 banks (FB1: the low bits of n2b, BLKC = 16 or 8 mod 32; FB2: the high bits of kap), so that
    // the 64-bit accesses of a half-warp stay conflict-free.
    constexpr int LB = NR == 8 ? 3 : 2, HB = 4 - LB;         // lane bits of n3l; high bits of kap taken from the lane index
    if (FWD) {
        __syncthreads();
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int c = tid + TC * i, n2b = (c >> LB) & (RB2 - 1), kap = c >> 6;
            Tw2 tw[8];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const float4 f = __ldg(&g_tab.fb1_c[LOGM - 15][kap][e]);
                tw[e] = Tw2{pack(f.x, f.y), pack(f.z, f.w)};
            }
            const int o = n2b * BLKC + n3l * ROW + 2 * kap;
            C2 v[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) v[brev<8>(r)] = lds2(re, im, o + r * RB2 * BLKC);
            dit8<false>(v, tw);
#pragma unroll
            for (int q = 0; q < 8; ++q) sts2(re, im, o + q * RB2 * BLKC, v[q]);
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < 16 / RB2; ++i) {
            const int c = tid + TC * i, k2a = (c >> 4) & 7;
            const int kap = (((c >> LB) & ((1 << HB) - 1)) << (4 - HB)) | ((c >> 7) & ((1 << (4 - HB)) - 1));
            Tw2 tw[8];
#pragma unroll
            for (int e = 0; e < RB2 / 2; ++e) {
                const float4 f = __ldg(&g_tab.fb2_c[LOGM - 15][8 * kap + k2a][e]);
                tw[e] = Tw2{pack(f.x, f.y), pack(f.z, f.w)};
            }
            const int o = k2a * RB2 * BLKC + n3l * ROW + 2 * kap;
            C2 v[RB2];
#pragma unroll
            for (int r = 0; r < RB2; ++r) v[brev<RB2>(r)] = lds2(re, im, o + r * BLKC);
            dit_r<RB2, false, Tw2, true>(v, tw);             // k2b >= RB2/2 (klow >= KL/2) stored conjugated
            if (kap == 0 && k2a == 0) column_factor(v[RB2 / 2]);      // column KL/2: k1 = 0, k2a = 0, k2b = RB2/2
#pragma unroll
            for (int q = 0; q < RB2; ++q) sts2(re, im, o + q * BLKC, v[q]);
        }
    }
    } else {
    // ---- n = 32768: FB1 radix 4 over n2a (4 butterflies per thread), FB2 radix 8 over n2b (2 per thread) ----
    // element (d2a, d2b, n3, k1) at (8 d2a + d2b) * BLK + n3 * ROW + k1
    if (FWD) {
        __syncthreads();
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int c = tid + T * i, n2b = (c >> 4) & 7, kap = c >> 7;
            Tw2 tw[8];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const float4 f = __ldg(&g_tab.fb1_14[kap][e]);
                tw[e] = Tw2{pack(f.x, f.y), pack(f.z, f.w)};
            }
            const int o = n2b * BLK + n3 * ROW + 2 * kap;
            C2 v[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) v[brev<4>(r)] = lds2(re, im, o + r * 8 * BLK);
            dit4<false>(v, tw);
#pragma unroll
            for (int q = 0; q < 4; ++q) sts2(re, im, o + q * 8 * BLK, v[q]);
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int c = tid + T * i, k2a = (c >> 4) & 3, kap = c >> 6;
            Tw2 tw[8];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const float4 f = __ldg(&g_tab.fb2_14[4 * kap + k2a][e]);
                tw[e] = Tw2{pack(f.x, f.y), pack(f.z, f.w)};
            }
            const int o = k2a * 8 * BLK + n3 * ROW + 2 * kap;
            C2 v[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) v[brev<8>(r)] = lds2(re, im, o + r * BLK);
            dit8<false, Tw2, true>(v, tw);                   // k2b >= 4 (klow >= KL/2) stored conjugated
            if (kap == 0 && k2a == 0) column_factor(v[4]);   // column KL/2 = 512: k1 = 0, k2a = 0, k2b = 4
#pragma unroll
            for (int q = 0; q < 8; ++q) sts2(re, im, o + q * BLK, v[q]);
        }
    }
    }
    auto special_prepare = [&]() {
    if (sl >= 0 && sl <= 16) {
        float2 ia = make_float2(0.f, 0.f), ib = make_float2(0.f, 0.f);            // what the injection adds to 2 X[k], 2 X[M-k]
        if (MODE == MODE_HDET) {
            ia = make_float2(a.two_fs * sha.x, sl == 0 ? 0.f : a.two_fs * sha.y);
            ib = make_float2(a.two_fs * shb.x, sl == 0 ? 0.f : a.two_fs * shb.y);
        } else if (MODE == MODE_FUSED) {
            const float2 cc = make_float2(cre, cim);
            if (sin_a) ia = amplfi::cmul(sha, amplfi::cmul(cc, unit_phase(sk)));
            if (sin_b) ib = amplfi::cmul(shb, amplfi::cmul(cc, unit_phase(M - sk)));
        }
        const float2 w = twiddle<N>(sk);
        sx[sl][0] = make_float4(sfa, sfb, ia.x, ia.y);
        sx[sl][1] = make_float4(ib.x, ib.y, w.x, w.y);
        if (VIEWS == 2) sraw[sl] = make_float4(sha.x, sha.y, shb.x, shb.y);
    }
    };
    special_prepare();

    // ---- FC: radix 16 over n3; lane A klow = t, lane B klow = 512 - t ----
    const int ka = t, kb = (t == 0) ? KL / 2 : KL - t;
    // column klow = k1 + 32 k2 lives at d2 = k2 (n = 32768: klow = k1 + 32 k2a + 128 k2b at d2 = 8 k2a + k2b)
    // (clusters: klow = k1 + 32 k2a + 256 k2b at d2 = RB2 k2a + k2b, blocks of BLKC in each CTA)
    auto column = [](int klow) {
        if (CL > 1) return (RB2 * ((klow >> 5) & 7) + (klow >> 8)) * BLKC + (klow & 31);
        return (LOGM <= 13 ? (klow >> 5) : 8 * ((klow >> 5) & 3) + (klow >> 7)) * BLK + (klow & 31);
    };
    const int oa = column(ka), obb = column(kb);
    // Lane B works on the CONJUGATED column 512 - t (FB stored it so): conj Z[512 - t + 512 q] = sum_n3 conj(B[n3]) W^n3
    // w16^(-n3 (q + 1)) with lane A's own W = w8192^t, i.e. the same twiddles serve both lanes and lane B's outputs appear
    // conjugated and reversed: v[q] = (Z[t + 512 q] | conj Z[512 - t + 512 (15 - q)]) -- exactly the partner bin of lane A.
    // Thread 0's lane B holds the self-paired column 256: its inputs took the factor conj(w32^n3) in FB and its outputs sit at
    // v[q] = conj Z[256 + 512 ((16 - q) & 15)].
    C2 v[16];
    if (FWD) {
        Tw1 tw[8];
        pass_twiddles<M>((float)ka, tw);
        if constexpr (CL > 1) {
            cg::this_cluster().sync();                       // every CTA has stored its rows of the columns (and has started)
            // row n3 = NR c + l of a column sits in CTA c: NR rows from this CTA's planes, the others from the peers'
            with_rank([&](auto rk) {
                constexpr int RK = decltype(rk)::value;
#pragma unroll
                for (int c = 0; c < CL; ++c) {
                    const float* qr = c == RK ? re : peer_re(c);
                    const float* qi = c == RK ? im : peer_im(c);
#pragma unroll
                    for (int l = 0; l < NR; ++l) {
                        const int r = NR * c + l, o = l * ROW;
                        v[brev<16>(r)] = C2{pack(qr[oa + o], qr[obb + o]), pack(qi[oa + o], qi[obb + o])};
                    }
                }
            });
        } else {
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 16; ++r)
                v[brev<16>(r)] = C2{pack(re[oa + r * ROW], re[obb + r * ROW]), pack(im[oa + r * ROW], im[obb + r * ROW])};
        }
        dit16<false>(v, tw);
    } else {
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = C2{0ull, 0ull};
        if constexpr (CL > 1) cg::this_cluster().sync(); else __syncthreads();
    }

    ulonglong2* park = nullptr;
    if constexpr (VIEWS == 2) {
        park = reinterpret_cast<ulonglong2*>(a.out2 + (size_t)unit * N) + t;
#pragma unroll
        for (int q = 0; q < 16; ++q) park[q * T] = make_ulonglong2(v[q].r, v[q].i);
    }
#pragma unroll 1
    for (int view = 0; view < VIEWS; ++view) {              // (the body, down to the stores of I3, keeps its indentation)
    if (VIEWS == 2 && view == 1) {
        // second view: arrival time later by t_shift[b]; the S table and the operands of the self-paired bins again, then
        // the spectrum back from the row it was parked in.  (Every thread is past the last barrier of the first view, so
        // nobody reads the first view's constants any more; the barrier below also fences the planes, which slower threads
        // may still be reading in I3.)
        delta += a.t_shift[b] * (double)a.inv_tseg;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const ulonglong2 pv = __ldcg(park + q * T);
            v[q] = C2{pv.x, pv.y};
        }
        view_constants();
        if (sl >= 0 && sl <= 16) {                           // the injected terms with the new phase; filter values and twiddle stay
            const float4 r4 = sraw[sl];
            const float2 cc = make_float2(cre, cim);
            const float2 ia = sl == 0 ? make_float2(0.f, 0.f) : amplfi::cmul(make_float2(r4.x, r4.y), amplfi::cmul(cc, unit_phase(sk)));
            const float2 ib = sl == 0 ? make_float2(0.f, 0.f) : amplfi::cmul(make_float2(r4.z, r4.w), amplfi::cmul(cc, unit_phase(M - sk)));
            const float4 s0 = sx[sl][0], s1 = sx[sl][1];
            sx[sl][0] = make_float4(s0.x, s0.y, ia.x, ia.y);
            sx[sl][1] = make_float4(ib.x, ib.y, s1.z, s1.w);
        }
        __syncthreads();
        out = a.out2 + (size_t)unit * n_out;
    }
    // ---- a-7 inject, a-8 whiten + band-limit ----
    // v[k3] = (Z[t + 512 k3] | Z[512 - t + 512 k3]) = (A[k3] | B[k3]).  Unit w < 8 (u = 2w) works on the two bin pairs
    //   lane 0: k0 = t + 512 u <-> M - k0 : (A[u], B[15-u]),      lane 1: k1 = k0 + 512 <-> M - k1 : (A[u+1], B[14-u])
    // as the two lanes of packed arithmetic; the first and last steps of split/merge are scalar so that operands meet in
    // the right lanes without moves.  Operands come in the slot layout (spec_layout.cuh): one 16-byte request each for
    // the four filter values, the two first h0 values and the two second ones, one unit ahead of their use.
    {
        // cr/ci[q]: conj B[15 - q] on entry (lane B of FC), B[q] on exit (lane B of I1)
        float ar[16], ai[16], cr[16], ci[16], br[16], bi[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            unpack(v[q].r, ar[q], cr[q]);
            unpack(v[q].i, ai[q], ci[q]);
        }
        if (t == 0) {
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                sc[q] = make_float2(ar[q], ai[q]);
                sc[16 + q] = make_float2(cr[(16 - q) & 15], -ci[(16 - q) & 15]);
            }
        }
        const float2 wt = twiddle<N>(t);                     // w_N^t
        float2 cf = make_float2(0.f, 0.f), cs = make_float2(0.f, 0.f);
        if (MODE == MODE_FUSED) {
            const float2 et = unit_phase(t);
            const float2 cc = make_float2(cre, cim);
            cf = amplfi::cmul(cc, et);                                        // C e(t)
            cs = amplfi::cmul_conj(amplfi::cmul(cc, s_em), et);               // C e(M) conj(e(t))
        }
        struct PwOps { float4 f, hf, hs; };
        auto pw_load = [&](int w, PwOps& L) {
            L.f = __ldg(fsl + w * T);
            L.hf = L.hs = make_float4(0.f, 0.f, 0.f, 0.f);
            if (MODE == MODE_HDET) {
                const int k0 = t + KL * 2 * w, k1 = k0 + KL;
                L.hf = make_float4(__ldg(hsrc + 2 * k0), __ldg(hsrc + 2 * k1), __ldg(hsrc + 2 * k0 + 1), __ldg(hsrc + 2 * k1 + 1));
                L.hs = make_float4(__ldg(hsrc + 2 * (M - k0)), __ldg(hsrc + 2 * (M - k1)), __ldg(hsrc + 2 * (M - k0) + 1),
                                   __ldg(hsrc + 2 * (M - k1) + 1));
            } else if (MODE == MODE_FUSED) {
                if (need & (1u << w)) L.hf = __ldg(hsl + w * T);
                if (need & (256u << w)) L.hs = __ldg(hsl + (8 + w) * T);
            }
        };
        PwOps ops[8];
        pw_load(0, ops[0]);
#pragma unroll
        for (int w8 = 0; w8 < 8; ++w8) {
            if (w8 + 1 < 8) pw_load(w8 + 1, ops[w8 + 1]);
            const PwOps& L = ops[w8];
            const int u = 2 * w8;
            const u64 ff = pack(L.f.x, L.f.y), fs = pack(L.f.z, L.f.w);
            // split twiddles (w_N^k0 | w_N^k1) = w_N^t (w32^u | w32^(u+1))
            const u64 kr = pack(kCos32[u], kCos32[u + 1]), ki = pack(-kSin32[u], -kSin32[u + 1]);
            C2 w;
            w.r = fma2(bc(wt.x), kr, neg2(mul2(bc(wt.y), ki)));
            w.i = fma2(bc(wt.x), ki, mul2(bc(wt.y), kr));
            // split: e = za + conj(zb), dd = za - conj(zb), wo = (-i dd) w, xa = e + wo, xb = conj(e - wo)
            const C2 e = C2{pack(ar[u] + cr[u], ar[u + 1] + cr[u + 1]), pack(ai[u] + ci[u], ai[u + 1] + ci[u + 1])};
            const C2 dd = C2{pack(ar[u] - cr[u], ar[u + 1] - cr[u + 1]), pack(ai[u] - ci[u], ai[u + 1] - ci[u + 1])};
            const C2 wo = C2{fma2(dd.i, w.r, mul2(dd.r, w.i)), fma2(dd.i, w.i, neg2(mul2(dd.r, w.r)))};
            C2 xa = C2{add2(e.r, wo.r), add2(e.i, wo.i)};
            C2 xb = C2{sub2(e.r, wo.r), sub2(wo.i, e.i)};
            if (MODE == MODE_HDET) {
                const u64 tf = bc(a.two_fs);
                xa.r = fma2(tf, pack(L.hf.x, L.hf.y), xa.r);
                xa.i = fma2(tf, pack(L.hf.z, L.hf.w), xa.i);
                xb.r = fma2(tf, pack(L.hs.x, L.hs.y), xb.r);
                xb.i = fma2(tf, pack(L.hs.z, L.hs.w), xb.i);
            } else if (MODE == MODE_FUSED) {
                if (need & (0x101u << w8)) {                 // warp-uniform
                    const float4 s4 = sp[w8];
                    const C2 spk = C2{pack(s4.x, s4.y), pack(s4.z, s4.w)};
                    if (need & (1u << w8)) {
                        const C2 h = C2{pack(L.hf.x, L.hf.y), pack(L.hf.z, L.hf.w)};
                        // PF = C e(t) (S[u] | S[u+1])
                        const C2 p = C2{fma2(bc(cf.x), spk.r, neg2(mul2(bc(cf.y), spk.i))), fma2(bc(cf.x), spk.i, mul2(bc(cf.y), spk.r))};
                        xa.r = fma2(h.r, p.r, fma2(neg2(h.i), p.i, xa.r));
                        xa.i = fma2(h.r, p.i, fma2(h.i, p.r, xa.i));
                    }
                    if (need & (256u << w8)) {
                        const C2 h = C2{pack(L.hs.x, L.hs.y), pack(L.hs.z, L.hs.w)};
                        // PS = C e(M) conj(e(t)) conj(S[u] | S[u+1])
                        const C2 p = C2{fma2(bc(cs.x), spk.r, mul2(bc(cs.y), spk.i)), fma2(bc(cs.y), spk.r, neg2(mul2(bc(cs.x), spk.i)))};
                        xb.r = fma2(h.r, p.r, fma2(neg2(h.i), p.i, xb.r));
                        xb.i = fma2(h.r, p.i, fma2(h.i, p.r, xb.i));
                    }
                }
            }
            xa.r = mul2(xa.r, ff); xa.i = mul2(xa.i, ff);
            xb.r = mul2(xb.r, fs); xb.i = mul2(xb.i, fs);
            // merge: e' = ya + conj(yb), d' = ya - conj(yb), o = d' conj(w), za' = e' + i o, zb' = conj(e') + i conj(o)
            const C2 e2 = C2{add2(xa.r, xb.r), sub2(xa.i, xb.i)};
            const C2 d2 = C2{sub2(xa.r, xb.r), add2(xa.i, xb.i)};
            const C2 o = C2{fma2(d2.r, w.r, mul2(d2.i, w.i)), fma2(d2.i, w.r, neg2(mul2(d2.r, w.i)))};
            float e0r, e1r, e0i, e1i, o0r, o1r, o0i, o1i;
            unpack(e2.r, e0r, e1r);
            unpack(e2.i, e0i, e1i);
            unpack(o.r, o0r, o1r);
            unpack(o.i, o0i, o1i);
            // lane 0: za' -> A[u], zb' -> B[15-u];  lane 1: za' -> A[u+1], zb' -> B[14-u]
            ar[u] = e0r - o0i;      ai[u] = e0i + o0r;      br[15 - u] = e0r + o0i; bi[15 - u] = o0r - e0i;
            ar[u + 1] = e1r - o1i;  ai[u + 1] = e1i + o1r;  br[14 - u] = e1r + o1i; bi[14 - u] = o1r - e1i;
        }
#pragma unroll
        for (int q = 0; q < 16; ++q) v[q] = C2{pack(ar[q], br[q]), pack(ai[q], bi[q])};
        // ---- the self-paired butterflies klow = 0 (lane A) and 256 (lane B) of thread 0, on 17 lanes of warp 0 ----
        // lane 0: Z[0];  lanes 1..7: (A[l], A[16-l]);  lane 8: A[8] with itself;  lanes 9..16: (B[q], B[15-q]), q = l - 9;
        // operands from sx (prepared after pass FB)
        if (t < 32) {
            __syncwarp();
            if (t <= 16) {
                const float4 s0 = sx[t][0], s1 = sx[t][1];
                if (t == 0) {       // Z[0] carries the DC and Nyquist bins of the real transform
                    const float2 z0 = sc[0];
                    const float x0 = 2.0f * (z0.x + z0.y) + s0.z, xm = 2.0f * (z0.x - z0.y) + s1.x;
                    const float y0 = x0 * s0.x, ym = xm * s0.y;
                    sc[0] = make_float2(y0 + ym, y0 - ym);
                } else {
                    const int ia = t <= 8 ? t : 7 + t, ib = t <= 8 ? 16 - t : 40 - t;
                    float2 pa = sc[ia], pb = sc[ib];
                    const float2 w = make_float2(s1.z, s1.w);
                    float2 xa, xb;
                    split_pair(pa, pb, w, xa, xb);
                    if (MODE != MODE_NONE) { xa.x += s0.z; xa.y += s0.w; xb.x += s1.x; xb.y += s1.y; }
                    // (explicitly rounded products: the result must not depend on how a MODE's surrounding code was contracted)
                    xa.x = __fmul_rn(xa.x, s0.x); xa.y = __fmul_rn(xa.y, s0.x); xb.x = __fmul_rn(xb.x, s0.y); xb.y = __fmul_rn(xb.y, s0.y);
                    merge_pair(xa, xb, w, pa, pb);
                    sc[ia] = pa;
                    if (ib != ia) sc[ib] = pb;
                }
            }
            __syncwarp();
            if (t == 0) {
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    const float2 pa = sc[q], pb = sc[16 + q];
                    v[q] = C2{pack(pa.x, pb.x), pack(pa.y, pb.y)};
                }
            }
        }
    }

    // ---- I1: inverse radix 16 over k3 ----
    {
        C2 w[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) w[brev<16>(r)] = v[r];
        dit16_const<true>(w);
        if constexpr (CL > 1) {
            with_rank([&](auto rk) {
                constexpr int RK = decltype(rk)::value;
#pragma unroll
                for (int c = 0; c < CL; ++c) {
                    float* qr = c == RK ? re : peer_re(c);
                    float* qi = c == RK ? im : peer_im(c);
#pragma unroll
                    for (int l = 0; l < NR; ++l) {
                        float ar, br, ai, bi;
                        unpack(w[NR * c + l].r, ar, br);
                        unpack(w[NR * c + l].i, ai, bi);
                        qr[oa + l * ROW] = ar; qi[oa + l * ROW] = ai;
                        qr[obb + l * ROW] = br; qi[obb + l * ROW] = bi;
                    }
                }
            });
        } else {
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            float ar, br, ai, bi;
            unpack(w[q].r, ar, br);
            unpack(w[q].i, ai, bi);
            re[oa + q * ROW] = ar; im[oa + q * ROW] = ai;
            re[obb + q * ROW] = br; im[obb + q * ROW] = bi;
        }
        }
    }
    if constexpr (LOGM <= 13) {
    // ---- I2: inverse radix RB over k2 (NB butterflies per thread; the twiddles depend on n3 only) ----
    {
        Tw1 tw[8];
#pragma unroll
        for (int e = 0; e < (RB == 16 ? 8 : (RB == 8 ? 4 : 2)); ++e) {
            const float2 f = __ldg(&g_tab.i2[LOGM - 11][n3][e]);
            tw[e] = Tw1{f.x, f.y};
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int ob = ob_of(i);
            C2 w[RB];
#pragma unroll
            for (int r = 0; r < RB; ++r) w[brev<RB>(r)] = lds2(re, im, ob + r * BLK);
            dit_r<RB, true>(w, tw);
#pragma unroll
            for (int q = 0; q < RB; ++q) sts2(re, im, ob + q * BLK, w[q]);
        }
    }
    } else if constexpr (CL > 1) {
    // ---- clusters: I2b inverse radix RB2 over k2b (twiddles by n3), I2a inverse radix 8 over k2a (twiddles by n3, n2b) ----
    {
        constexpr int LB = NR == 8 ? 3 : 2, HB = 4 - LB;
        Tw1 tw[8];
#pragma unroll
        for (int e = 0; e < RB2 / 2; ++e) {
            const float2 f = __ldg(&g_tab.i2b_c[LOGM - 15][n3][e]);
            tw[e] = Tw1{f.x, f.y};
        }
        cg::this_cluster().sync();                           // the peers' I1 results have arrived
#pragma unroll
        for (int i = 0; i < 16 / RB2; ++i) {
            const int c = tid + TC * i, k2a = (c >> 4) & 7;
            const int kap = (((c >> LB) & ((1 << HB) - 1)) << (4 - HB)) | ((c >> 7) & ((1 << (4 - HB)) - 1));
            const int o = k2a * RB2 * BLKC + n3l * ROW + 2 * kap;
            C2 w[RB2];
#pragma unroll
            for (int r = 0; r < RB2; ++r) w[brev<RB2>(r)] = lds2(re, im, o + r * BLKC);
            dit_r<RB2, true>(w, tw);
#pragma unroll
            for (int q = 0; q < RB2; ++q) sts2(re, im, o + q * BLKC, w[q]);
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int c = tid + TC * i, n2b = (c >> LB) & (RB2 - 1), kap = c >> 6;
            Tw1 ta[8];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const float2 f = __ldg(&g_tab.i2a_c[LOGM - 15][16 * n2b + n3][e]);
                ta[e] = Tw1{f.x, f.y};
            }
            const int o = n2b * BLKC + n3l * ROW + 2 * kap;
            C2 w[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) w[brev<8>(r)] = lds2(re, im, o + r * RB2 * BLKC);
            dit8<true>(w, ta);
#pragma unroll
            for (int q = 0; q < 8; ++q) sts2(re, im, o + q * RB2 * BLKC, w[q]);
        }
    }
    } else {
    // ---- n = 32768: I2b inverse radix 8 over k2b (twiddles by n3), I2a inverse radix 4 over k2a (twiddles by n3, n2b) ----
    {
        Tw1 tw[8];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float2 f = __ldg(&g_tab.i2b_14[n3][e]);
            tw[e] = Tw1{f.x, f.y};
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int c = tid + T * i, k2a = (c >> 4) & 3, kap = c >> 6;
            const int o = k2a * 8 * BLK + n3 * ROW + 2 * kap;
            C2 w[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) w[brev<8>(r)] = lds2(re, im, o + r * BLK);
            dit8<true>(w, tw);
#pragma unroll
            for (int q = 0; q < 8; ++q) sts2(re, im, o + q * BLK, w[q]);
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int c = tid + T * i, n2b = (c >> 4) & 7, kap = c >> 7;
            Tw1 ta[8];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const float2 f = __ldg(&g_tab.i2a_14[16 * n2b + n3][e]);
                ta[e] = Tw1{f.x, f.y};
            }
            const int o = n2b * BLK + n3 * ROW + 2 * kap;
            C2 w[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) w[brev<4>(r)] = lds2(re, im, o + r * 8 * BLK);
            dit4<true>(w, ta);
#pragma unroll
            for (int q = 0; q < 4; ++q) sts2(re, im, o + q * 8 * BLK, w[q]);
        }
    }
    }
    // ---- I3: inverse radix 32 over k1, natural-order stores ----
    {
        const float jf = (float)j;
        Tw1 tw[8];
        pass_twiddles<M>(2.0f * jf, tw);                     // base W^2, W = w_M^j
        __syncthreads();
        C2 w[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) w[brev<16>(r)] = lds2(re, im, oj + 2 * r);
        dit16<true>(w, tw);
        float2* out2 = reinterpret_cast<float2*>(out);
        constexpr float uu = -6.283185307179586f / (float)M;
        const int c2 = a.crop >> 1;                          // crop is even: whole float2 pairs
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            float er, orr, ei, oi;
            unpack(w[q].r, er, orr);
            unpack(w[q].i, ei, oi);
            const Tw1 tq = tan_twiddle(fmaf(jf, uu, (float)(M / 32 * (q & 7)) * uu));      // W w32^q (the +i of q >= 8 as ROT)
            float2 lo, hi;
            if (q < 8) bf_s<true, false>(make_float2(er, ei), make_float2(orr, oi), tq, lo, hi);
            else bf_s<true, true>(make_float2(er, ei), make_float2(orr, oi), tq, lo, hi);
            const int m0 = q * T + j, m1 = (q + 16) * T + j;
            if (a.crop == 0) {
                __stcs(out2 + m0, lo);
                __stcs(out2 + m1, hi);
            } else {
                if (m0 >= c2 && m0 < M - c2) __stcs(out2 + m0 - c2, lo);
                if (m1 >= c2 && m1 < M - c2) __stcs(out2 + m1 - c2, hi);
            }
        }
    }
    }   // views
}

__global__ void init_tables3_kernel() {
    // one thread per (segment length lg, row, entry): rows in the layout fft_tan.cuh gives each radix
    //   RB = 16: W^8, W^4, W^2, W^2 w8, W w16^q (q < 4);   RB = 8: W^4, W^2, W w8^q (q < 2);   RB = 4: W^2, W
    const int i = threadIdx.x;                                 // 0 .. 383
    if (i >= 384) return;
    const int lg = i >> 7, row = (i >> 3) & 15, ent = i & 7;
    const int m = 2048 << lg, rb = m / 512;
    auto ct = [m](int e, float& c, float& tau) {               // (c, tau) of w_M^e, fp64 -> fp32
        double s, co;
        sincospi(-2.0 * (double)(e & (m - 1)) / (double)m, &s, &co);
        if (fabs(co) < 1e-12) co = 1e-12;
        c = (float)co;
        tau = (float)(s / co);
    };
    auto expo = [m, rb](int x, int ent) {                      // exponent of entry `ent` for W = w_M^x
        if (rb == 16) {
            switch (ent) {
                case 0: return 8 * x;
                case 1: return 4 * x;
                case 2: return 2 * x;
                case 3: return 2 * x + m / 8;
                default: return x + m / 16 * (ent - 4);
            }
        }
        if (rb == 8) {
            switch (ent) {
                case 0: return 4 * x;
                case 1: return 2 * x;
                default: return x + m / 8 * ((ent - 2) & 1);
            }
        }
        return ent == 0 ? 2 * x : x;
    };
    float4 f;
    ct(expo(16 * (2 * row), ent), f.x, f.z);                   // FB lane A: W = w_(32 RB)^(2 kap) = w_M^(32 kap)
    ct(expo(16 * (2 * row + 1), ent), f.y, f.w);               // lane B: k1 = 2 kap + 1
    g_tab.fb[lg][row][ent] = f;
    float2 g;
    ct(expo(32 * row, ent), g.x, g.y);                         // I2: W = w_(16 RB)^n3 = w_M^(32 n3)
    g_tab.i2[lg][row][ent] = g;
}

// n = 32768 (M = 16384): radix-4 rows (W^2, W) and radix-8 rows (W^4, W^2, W, W w8)
__global__ void init_tables3_14_kernel() {
    constexpr int m = 16384;
    auto ct = [](int e, float& c, float& tau) {
        double s, co;
        sincospi(-2.0 * (double)(e & (m - 1)) / (double)m, &s, &co);
        if (fabs(co) < 1e-12) co = 1e-12;
        c = (float)co;
        tau = (float)(s / co);
    };
    auto e4 = [](int x, int ent) { return ent == 0 ? 2 * x : x; };
    auto e8 = [](int x, int ent) { return ent == 0 ? 4 * x : (ent == 1 ? 2 * x : x + m / 8 * (ent - 2)); };
    const int i = blockIdx.x * blockDim.x + threadIdx.x;       // 0 .. 511
    if (i < 32) {                                              // fb1: W = w_128^k1 = w_M^(128 k1), lanes k1 = 2 kap, 2 kap + 1
        const int kap = i >> 1, ent = i & 1;
        float4 f;
        ct(e4(128 * (2 * kap), ent), f.x, f.z);
        ct(e4(128 * (2 * kap + 1), ent), f.y, f.w);
        g_tab.fb1_14[kap][ent] = f;
    }
    if (i < 256) {                                             // fb2: W = w_1024^(k1 + 32 k2a) = w_M^(16 (k1 + 32 k2a))
        const int row = i >> 2, ent = i & 3, kap = row >> 2, k2a = row & 3;
        float4 f;
        ct(e8(16 * (2 * kap + 32 * k2a), ent), f.x, f.z);
        ct(e8(16 * (2 * kap + 1 + 32 * k2a), ent), f.y, f.w);
        g_tab.fb2_14[row][ent] = f;
        const int row2 = i >> 1, ent2 = i & 1;                  // i2a: W = w_512^(n3 + 16 n2b) = w_M^(32 row), row = 16 n2b + n3
        float2 g;
        ct(e4(32 * row2, ent2), g.x, g.y);
        g_tab.i2a_14[row2][ent2] = g;
    }
    if (i < 64) {                                              // i2b: W = w_128^n3 = w_M^(128 n3)
        const int n3 = i >> 2, ent = i & 3;
        float2 g;
        ct(e8(128 * n3, ent), g.x, g.y);
        g_tab.i2b_14[n3][ent] = g;
    }
}

// clusters (n = 65536, 131072; lg = 0, 1): the four middle-pass tables; radix-8 rows (W^4, W^2, W, W w8), radix-16 rows as in
// pass_twiddles (W^8, W^4, W^2, W^2 w8, W w16^q)
__global__ void init_tables3_cluster_kernel() {
    const int lg = blockIdx.y;                                 // 0: M = 32768 (RB2 = 8), 1: M = 65536 (RB2 = 16)
    const int m = 32768 << lg, rb2 = 8 << lg;
    auto ct = [m](int e, float& c, float& tau) {
        double s, co;
        sincospi(-2.0 * (double)(e & (m - 1)) / (double)m, &s, &co);
        if (fabs(co) < 1e-12) co = 1e-12;
        c = (float)co;
        tau = (float)(s / co);
    };
    auto e8 = [m](int x, int ent) { return ent == 0 ? 4 * x : (ent == 1 ? 2 * x : x + m / 8 * (ent - 2)); };
    auto e16 = [m](int x, int ent) {
        switch (ent) {
            case 0: return 8 * x;
            case 1: return 4 * x;
            case 2: return 2 * x;
            case 3: return 2 * x + m / 8;
            default: return x + m / 16 * (ent - 4);
        }
    };
    const int i = blockIdx.x * blockDim.x + threadIdx.x;       // 0 .. 2047
    const int row = i >> 3, ent = i & 7;                       // row 0 .. 255
    if (row < 16 && ent < 4) {                                 // fb1: W = w_256^k1 = w_M^((M/256) k1), lanes k1 = 2 kap, 2 kap + 1
        float4 f;
        ct(e8((m / 256) * (2 * row), ent), f.x, f.z);
        ct(e8((m / 256) * (2 * row + 1), ent), f.y, f.w);
        g_tab.fb1_c[lg][row][ent] = f;
    }
    if (row < 16 && ent < rb2 / 2) {                           // i2b: W = w_(M/256)^n3 = w_M^(256 n3), radix rb2
        float2 g;
        const int x = 256 * row;
        ct(rb2 == 8 ? e8(x, ent) : e16(x, ent), g.x, g.y);
        g_tab.i2b_c[lg][row][ent] = g;
    }
    if (row < 128 && ent < rb2 / 2) {                          // fb2: W = w_(M/16)^(k1 + 32 k2a), row = 8 kap + k2a, radix rb2
        const int kap = row >> 3, k2a = row & 7;
        const int xa = 16 * (2 * kap + 32 * k2a), xb = 16 * (2 * kap + 1 + 32 * k2a);
        float4 f;
        ct(rb2 == 8 ? e8(xa, ent) : e16(xa, ent), f.x, f.z);
        ct(rb2 == 8 ? e8(xb, ent) : e16(xb, ent), f.y, f.w);
        g_tab.fb2_c[lg][row][ent] = f;
    }
    if (row < 16 * rb2 && ent < 4) {                           // i2a: W = w_M^(32 (n3 + 16 n2b)), row = 16 n2b + n3, radix 8
        float2 g;
        ct(e8(32 * row, ent), g.x, g.y);
        g_tab.i2a_c[lg][row][ent] = g;
    }
}

}  // namespace v3

// Once per device (amplfi_plan_create synchronises before it returns).
int init_iw3_tables(cudaStream_t st) {
    static std::atomic<unsigned> done{0};
    int dev = 0;
    cudaGetDevice(&dev);
    const unsigned bit = 1u << (dev & 31);
    if (done.load(std::memory_order_acquire) & bit) return AMPLFI_OK;
    v3::init_tables3_kernel<<<1, 384, 0, st>>>();
    v3::init_tables3_14_kernel<<<1, 256, 0, st>>>();
    v3::init_tables3_cluster_kernel<<<dim3(8, 2), 256, 0, st>>>();
    count_launch(3);
    const int rc = check_launch("init_tables3_kernel");
    if (rc) return rc;
    if (cudaStreamSynchronize(st) != cudaSuccess) { set_error("init_tables3_kernel: synchronise failed"); return AMPLFI_ERR_CUDA; }
    done.fetch_or(bit, std::memory_order_release);
    return AMPLFI_OK;
}

template <int LOGM, int MODE, bool FWD, int VIEWS = 1>
static int launch_iw3_t(const IwArgs& a, int units, cudaStream_t st) {
    using G = v3::Geo<LOGM>;
    static std::atomic<unsigned> attr_done{0};
    const int rc = ensure_dynamic_smem(v3::inject_whiten3_kernel<LOGM, MODE, FWD, VIEWS>, G::SMEM_BYTES, attr_done);
    if (rc) return rc;
    if constexpr (G::CL == 1) {
        v3::inject_whiten3_kernel<LOGM, MODE, FWD, VIEWS><<<units, G::TC, G::SMEM_BYTES, st>>>(a, units);
    } else {                        // one cluster of G::CL CTAs per unit
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)units * G::CL);
        cfg.blockDim = dim3(G::TC);
        cfg.dynamicSmemBytes = G::SMEM_BYTES;
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = G::CL;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        const cudaError_t e = cudaLaunchKernelEx(&cfg, v3::inject_whiten3_kernel<LOGM, MODE, FWD>, a, units);
        if (e != cudaSuccess) { set_error("inject_whiten3_kernel: cluster launch: %s", cudaGetErrorString(e)); return AMPLFI_ERR_CUDA; }
    }
    count_launch();
    return check_launch("inject_whiten3_kernel");
}

template <int LOGM>
static int launch_iw3_l(const IwArgs& a, int mode, int units, cudaStream_t st) {
    if (a.out2 != nullptr) {        // two data views from one forward transform
        if constexpr (LOGM <= 13) {
            if (mode != MODE_FUSED || a.noise == nullptr || a.t_shift == nullptr || a.crop != 0 || (reinterpret_cast<size_t>(a.out2) & 15)) {
                set_error("inject_whiten3: the two-view launch needs the fused mode and a 16-byte aligned second output");
                return AMPLFI_ERR_INVALID_ARG;
            }
            return launch_iw3_t<LOGM, MODE_FUSED, true, 2>(a, units, st);
        } else {
            set_error("inject_whiten3: no two-view launch for this segment length");
            return AMPLFI_ERR_UNSUPPORTED_SIZE;
        }
    }
    if (a.noise == nullptr) {       // inverse-only launches (time-domain waveform, filter design)
        if (mode == MODE_HDET) return launch_iw3_t<LOGM, MODE_HDET, false>(a, units, st);
        if (mode == MODE_FUSED) return launch_iw3_t<LOGM, MODE_FUSED, false>(a, units, st);
        set_error("inject_whiten3: no data and nothing to inject");
        return AMPLFI_ERR_INVALID_ARG;
    }
    switch (mode) {
        case MODE_NONE: return launch_iw3_t<LOGM, MODE_NONE, true>(a, units, st);
        case MODE_HDET: return launch_iw3_t<LOGM, MODE_HDET, true>(a, units, st);
        default: return launch_iw3_t<LOGM, MODE_FUSED, true>(a, units, st);
    }
}

int launch_iw3(const IwArgs& a, int logm, int mode, int units, cudaStream_t st) {
    if (logm == 16) return launch_iw3_l<16>(a, mode, units, st);
    if (logm == 15) return launch_iw3_l<15>(a, mode, units, st);
    if (logm == 14) return launch_iw3_l<14>(a, mode, units, st);
    if (logm == 13) return launch_iw3_l<13>(a, mode, units, st);
    if (logm == 12) return launch_iw3_l<12>(a, mode, units, st);
    return launch_iw3_l<11>(a, mode, units, st);
}

}  // namespace amplfi
