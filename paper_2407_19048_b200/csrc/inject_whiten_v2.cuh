// inject_whiten_v2.cuh -- second-generation fused kernel for N = 16384 (M = 8192 complex points):
// four passes 16 * 8 * 8 * 8, 16 points per thread, 512 threads per segment, packed fp32x2 arithmetic.
//
// Index algebra.  Input index  n = n1*512 + n2*64 + n3*8 + n4   (n1 < 16, n2, n3, n4 < 8)
//                 output bin   k = k1 + 16*k2 + 128*k3 + 1024*k4 (k1 < 16, k2, k3, k4 < 8)
//   P1 (radix 16 over n1, operands from global memory): one scalar radix-2 stage over the top bit of n1
//       splits the butterfly into the even-k1 and odd-k1 halves, which then run as ONE packed radix-8
//       (half A = even k1 = 2*kap, half B = odd k1 = 2*kap + 1).  Twiddle w_M^(j1 k1), j1 = n2*64+n3*8+n4.
//   P2 (packed radix 8 over n2), twiddle w_512^((n3*8+n4) k2); both halves share it.
//   P3 (packed radix 8 over n3), twiddle w_64^(n4 k3).
//   P4 (packed radix 8 over n4): half A is the butterfly with klow = k1+16k2+128k3 = t, half B the one with
//       klow' = 1024 - t, so bins k and M - k meet in one thread: split / inject / whiten / merge in registers.
//   The inverse runs P4' P3' P2' P1' with conjugate twiddles and stores natural-order samples.
//
// Shared memory: two float planes (re, im) of M floats.  Float index of element (kap, pi, d2, d3, d4) is
//   pi + 2*slot,  slot = kap<<9 | d2<<6 | (d3>>1)<<4 | ((d4 ^ kap) & 7)<<1 | ((d3 ^ d2) & 1)
// so that the 64-bit (A, B) accesses of P1..P3 and the 32-bit accesses of P4 are all bank-conflict free.
#pragma once
#include "fft_packed.cuh"
#include "waveform.cuh"

namespace amplfi {
namespace v2 {

using namespace pk;

constexpr int M13 = 8192, N13 = 16384, T13 = 512;

// Geometry of the two supported lengths.  LOGM = 13: M = 8192 = 16*8*8*8 (N = 16384, the index algebra above).
// LOGM = 12: M = 4096 = 8*8*8*8 (N = 8192, the paper's own 4 s at 2048 Hz): pass 1 is a radix 8 and every
// virtual thread takes two of its butterflies (j1 = t and t + 256); passes 2-4 are unchanged with kap < 4.
// LOGM = 11: M = 2048 = 4*8*8*8 (N = 4096): pass 1 is a radix 4, four butterflies per virtual thread (j1 = t + 128 h), kap < 2.
template <int LOGM>
struct Geo {
    static constexpr int M = 1 << LOGM, N = 2 * M;
    static constexpr int R1 = M / 512;                 // radix of pass 1: 16 or 8
    static constexpr int LR1 = LOGM - 9;               // log2 R1
    static constexpr int T = M / 16;                   // virtual threads: 512 or 256
    static constexpr int KL = 64 * R1;                 // span of klow = k1 + R1 k2 + 8 R1 k3: 1024 or 512
    static constexpr int S3 = LR1 + 3;                 // klow >> S3 = k3
};
// complex index (in float2 units) of the i-th of the 16 samples of virtual thread t
template <int LOGM>
__device__ __forceinline__ int sample_index(int i, int t) {
    if constexpr (LOGM == 13) return i * 512 + t;
    else return (i & (Geo<LOGM>::R1 - 1)) * 512 + t + Geo<LOGM>::T * (i >> Geo<LOGM>::LR1);
}

__device__ __forceinline__ int slot13(int kap, int d2, int d3, int d4) {
    return (kap << 9) | (d2 << 6) | ((d3 >> 1) << 4) | (((d4 ^ kap) & 7) << 1) | ((d3 ^ d2) & 1);
}
__device__ __forceinline__ C2 lds2(const float* re, const float* im, int slot) {
    return C2{*reinterpret_cast<const u64*>(re + 2 * slot), *reinterpret_cast<const u64*>(im + 2 * slot)};
}
__device__ __forceinline__ void sts2(float* re, float* im, int slot, C2 v) {
    *reinterpret_cast<u64*>(re + 2 * slot) = v.r;
    *reinterpret_cast<u64*>(im + 2 * slot) = v.i;
}

// ---- twiddle tables of the passes whose twiddles depend on few index bits (filled once by init_tw13, fp64 -> fp32) ----
//   p2[q][s]  = (g[2q], g[2q+1]),  g[k] = w_512^(s k),              s = n3*8 + n4      (P2 forward)
//   p3[q][s]  = (g[2q], g[2q+1]),  g[k] = w_64^(s k),               s = n4             (P3 forward)
//   p3i[q][s] = (g[2q], g[2q+1]),  g[n3] = w_512^((n3*8 + n4) k2),  s = k2*8 + n4      (P3 inverse: conj twiddle of P2)
//   p4i[c][n4] = halves (w_64^(n4 k3a), w_64^(n4 k3b)) in the packed layout, c = the (k3a, k3b) combination of thread t
// 9.5 KB, read through L1 by every CTA; the twiddles of P1 forward / P2 inverse depend on all nine bits of t (64 KB per
// table) and stay computed.
struct Tw13 {
    float4 p2[4][64];
    float4 p3[4][8];
    float4 p3i[4][64];
    ulonglong2 p4i[3][8][8];      // [LOGM - 11]
};
static __device__ Tw13 g_tw13;       // this header is included by inject_whiten13.cu only

__device__ __forceinline__ void tw_load8(const float4* col, int stride, float2 (&g)[8]) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float4 f = __ldg(col + q * stride);
        g[2 * q] = make_float2(f.x, f.y);
        g[2 * q + 1] = make_float2(f.z, f.w);
    }
}

// ---- forward passes ----
// x[n1] = z[n1*512 + t] (natural complex, from global).  Leaves the spectrum digits (k1; n2 n3 n4) in smem.
// dif4 / dit4: the last two stages of dif8 / the first two of dit8, on four packed elements
__device__ __forceinline__ void dif4(C2 (&v)[4]) {
    C2 d;
    d = csub(v[0], v[2]); v[0] = cadd(v[0], v[2]); v[2] = d;
    d = csub(v[1], v[3]); v[1] = cadd(v[1], v[3]); v[3] = mul_w8<2, false>(d);
    d = csub(v[0], v[1]); v[0] = cadd(v[0], v[1]); v[1] = d;
    d = csub(v[2], v[3]); v[2] = cadd(v[2], v[3]); v[3] = d;
}
__device__ __forceinline__ void dit4(C2 (&v)[4]) {
    C2 b;
    b = v[1]; v[1] = csub(v[0], b); v[0] = cadd(v[0], b);
    b = v[3]; v[3] = csub(v[2], b); v[2] = cadd(v[2], b);
    b = v[2]; v[2] = csub(v[0], b); v[0] = cadd(v[0], b);
    b = mul_w8<2, true>(v[3]); v[3] = csub(v[1], b); v[1] = cadd(v[1], b);
}

// M = 4096: x[h*8 + n1] = z[n1*512 + j1], j1 = t + 256 h.  Per butterfly: scalar radix-2 stage over the top bit of n1, then one
// packed radix 4 over the even-k1 / odd-k1 halves (k1 = 2 kap, 2 kap + 1, kap < 4); twiddle w_M^(j1 k1).
__device__ __forceinline__ void p1_fwd12(const float2 (&x)[16], int t, float* re, float* im) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int j1 = t + 256 * h;
        C2 v[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 s = amplfi::cadd(x[h * 8 + i], x[h * 8 + i + 4]);
            float2 d = amplfi::csub(x[h * 8 + i], x[h * 8 + i + 4]);
            switch (i) {      // d *= w8^i
                case 0: break;
                case 1: d = mul_w32<4, false>(d); break;
                case 2: d = mul_w32<8, false>(d); break;
                default: d = mul_w32<12, false>(d); break;
            }
            v[i] = C2{pack(s.x, d.x), pack(s.y, d.y)};
        }
        dif4(v);
        const float2 u = twiddle<4096>(j1);
        const float2 u2 = twiddle<4096>(2 * j1);
        const C2 base = C2{pack(1.0f, u.x), pack(0.0f, u.y)}, step = C2{bcast(u2.x), bcast(u2.y)};
        const C2 s2 = cmul(step, step);
        const C2 tw[4] = {base, cmul(base, step), cmul(base, s2), cmul(cmul(base, step), s2)};
        const int n2 = j1 >> 6, n3 = (j1 >> 3) & 7, n4 = j1 & 7;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int kap = brev<4>(r);
            sts2(re, im, slot13(kap, n2, n3, n4), cmul(v[r], tw[kap]));
        }
    }
}

// M = 2048: x[h*4 + n1] = z[n1*512 + j1], j1 = t + 128 h, h < 4.  Radix 4 = scalar radix-2 stage + packed radix 2.
__device__ __forceinline__ void p1_fwd11(const float2 (&x)[16], int t, float* re, float* im) {
#pragma unroll
    for (int h = 0; h < 4; ++h) {
        const int j1 = t + 128 * h;
        const float2 s0 = amplfi::cadd(x[h * 4], x[h * 4 + 2]), d0 = amplfi::csub(x[h * 4], x[h * 4 + 2]);
        const float2 s1 = amplfi::cadd(x[h * 4 + 1], x[h * 4 + 3]);
        const float2 d1 = mul_w32<8, false>(amplfi::csub(x[h * 4 + 1], x[h * 4 + 3]));       // * w4^1 = -i
        const C2 v0 = C2{pack(s0.x, d0.x), pack(s0.y, d0.y)}, v1 = C2{pack(s1.x, d1.x), pack(s1.y, d1.y)};
        const float2 u = twiddle<2048>(j1);
        const float2 u2 = twiddle<2048>(2 * j1);
        const C2 base = C2{pack(1.0f, u.x), pack(0.0f, u.y)}, step = C2{bcast(u2.x), bcast(u2.y)};
        const int n2 = j1 >> 6, n3 = (j1 >> 3) & 7, n4 = j1 & 7;
        sts2(re, im, slot13(0, n2, n3, n4), cmul(cadd(v0, v1), base));
        sts2(re, im, slot13(1, n2, n3, n4), cmul(csub(v0, v1), cmul(base, step)));
    }
}
__device__ __forceinline__ void p1_inv11(float2 (&x)[16], int t, const float* re, const float* im) {
#pragma unroll
    for (int h = 0; h < 4; ++h) {
        const int j1 = t + 128 * h;
        const int n2 = j1 >> 6, n3 = (j1 >> 3) & 7, n4 = j1 & 7;
        const C2 a = lds2(re, im, slot13(0, n2, n3, n4)), b = lds2(re, im, slot13(1, n2, n3, n4));
        const C2 v0 = cadd(a, b), v1 = csub(a, b);
        float2 s0, d0, s1, d1;
        unpack(v0.r, s0.x, d0.x); unpack(v0.i, s0.y, d0.y);
        unpack(v1.r, s1.x, d1.x); unpack(v1.i, s1.y, d1.y);
        d1 = mul_w32<8, true>(d1);                                                           // * conj(w4^1) = +i
        x[h * 4] = amplfi::cadd(s0, d0); x[h * 4 + 2] = amplfi::csub(s0, d0);
        x[h * 4 + 1] = amplfi::cadd(s1, d1); x[h * 4 + 3] = amplfi::csub(s1, d1);
    }
}

__device__ __forceinline__ void p1_fwd(const float2 (&x)[16], int t, float* re, float* im) {
    C2 v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float2 s = amplfi::cadd(x[i], x[i + 8]);
        float2 d = amplfi::csub(x[i], x[i + 8]);
        switch (i) {      // d *= w16^i
            case 0: break;
            case 1: d = mul_w32<2, false>(d); break;
            case 2: d = mul_w32<4, false>(d); break;
            case 3: d = mul_w32<6, false>(d); break;
            case 4: d = mul_w32<8, false>(d); break;
            case 5: d = mul_w32<10, false>(d); break;
            case 6: d = mul_w32<12, false>(d); break;
            default: d = mul_w32<14, false>(d); break;
        }
        v[i] = C2{pack(s.x, d.x), pack(s.y, d.y)};
    }
    dif8(v);
    // twiddles (w^(j1 2kap), w^(j1 (2kap+1))) = (1, u) * (u^2)^kap,  u = w_M^j1
    const float2 u = twiddle<M13>(t);
    const float2 u2 = twiddle<M13>(2 * t);
    C2 tw[8];
    powers8(C2{pack(1.0f, u.x), pack(0.0f, u.y)}, C2{bcast(u2.x), bcast(u2.y)}, tw);
    const int n2 = t >> 6, n3 = (t >> 3) & 7, n4 = t & 7;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int kap = brev<8>(r);
        sts2(re, im, slot13(kap, n2, n3, n4), cmul(v[r], tw[kap]));
    }
}

// g: the twiddle row of set t & 63 (tw_load8 of g_tw13.p2), requested by the caller ahead of the barrier
__device__ __forceinline__ void p2_fwd(int t, float* re, float* im, const float2 (&g)[8]) {
    const int kap = t >> 6, n3 = (t >> 3) & 7, n4 = t & 7;
    C2 v[8];
#pragma unroll
    for (int n2 = 0; n2 < 8; ++n2) v[n2] = lds2(re, im, slot13(kap, n2, n3, n4));
    dif8(v);
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int k2 = brev<8>(r);
        sts2(re, im, slot13(kap, k2, n3, n4), k2 == 0 ? v[r] : cmul_s(v[r], g[k2]));
    }
}

__device__ __forceinline__ void p3_fwd(int t, float* re, float* im, const float2 (&g)[8]) {
    const int kap = t >> 6, k2 = (t >> 3) & 7, n4 = t & 7;
    C2 v[8];
#pragma unroll
    for (int n3 = 0; n3 < 8; ++n3) v[n3] = lds2(re, im, slot13(kap, k2, n3, n4));
    dif8(v);
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int k3 = brev<8>(r);
        sts2(re, im, slot13(kap, k2, k3, n4), k3 == 0 ? v[r] : cmul_s(v[r], g[k3]));
    }
}

struct P4Addr { int fa, fb, xa, xb; };     // float offsets of halves A, B at d4 = 0 and their kap (xor masks)

template <int LOGM>
__device__ __forceinline__ void p4_addr(int klow, int& base, int& kap) {
    const int k1 = klow & (Geo<LOGM>::R1 - 1), k2 = (klow >> Geo<LOGM>::LR1) & 7, k3 = klow >> Geo<LOGM>::S3;
    kap = k1 >> 1;
    base = (k1 & 1) + 2 * ((kap << 9) | (k2 << 6) | ((k3 >> 1) << 4) | ((k3 ^ k2) & 1));
}
// element d4 of the butterfly at (base, kap): float index base + 2*(((d4 ^ kap) & 7) << 1)
__device__ __forceinline__ int p4_off(int base, int kap, int d4) { return base + (((d4 ^ kap) & 7) << 2); }

template <int LOGM>
__device__ __forceinline__ void p4_fwd(int klow_a, int klow_b, C2 (&v)[8], const float* re, const float* im) {
    int ba, ka, bb, kb;
    p4_addr<LOGM>(klow_a, ba, ka);
    p4_addr<LOGM>(klow_b, bb, kb);
#pragma unroll
    for (int n4 = 0; n4 < 8; ++n4) {
        const int oa = p4_off(ba, ka, n4), ob = p4_off(bb, kb, n4);
        v[n4] = C2{pack(re[oa], re[ob]), pack(im[oa], im[ob])};
    }
    dif8(v);
}

// ---- inverse passes ----
template <int LOGM>
__device__ __forceinline__ void p4_inv(int klow_a, int klow_b, C2 (&v)[8], float* re, float* im) {
    dit8(v);
    int ba, ka, bb, kb;
    p4_addr<LOGM>(klow_a, ba, ka);
    p4_addr<LOGM>(klow_b, bb, kb);
    // conj twiddle of P3: w_64^(-n4 k3) per half, from the table row of this thread's (k3a, k3b) combination
    constexpr int S3 = Geo<LOGM>::S3;
    const ulonglong2* trow = g_tw13.p4i[LOGM - 11][2 * (klow_a >> S3) + ((klow_a & ((1 << S3) - 1)) != 0 ? 1 : 0)];
#pragma unroll
    for (int n4 = 0; n4 < 8; ++n4) {
        C2 y = v[0];
        if (n4 != 0) {
            const ulonglong2 w = __ldg(trow + n4);
            y = cmul_conj(v[n4], C2{w.x, w.y});
        }
        float ar, br, ai, bi;
        unpack(y.r, ar, br);
        unpack(y.i, ai, bi);
        const int oa = p4_off(ba, ka, n4), ob = p4_off(bb, kb, n4);
        re[oa] = ar; im[oa] = ai;
        re[ob] = br; im[ob] = bi;
    }
}

__device__ __forceinline__ void p3_inv(int t, float* re, float* im, const float2 (&g)[8]) {
    const int kap = t >> 6, k2 = (t >> 3) & 7, n4 = t & 7;
    C2 v[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) v[r] = lds2(re, im, slot13(kap, k2, brev<8>(r), n4));
    dit8(v);
    // conj twiddle of P2: w_512^(-(n3*8 + n4) k2): g = row t & 63 of g_tw13.p3i
#pragma unroll
    for (int n3 = 0; n3 < 8; ++n3) sts2(re, im, slot13(kap, k2, n3, n4), cmul_conj_s(v[n3], g[n3]));
}

// conj twiddles of P1 for virtual thread t: w_M^(-(n2*64 + j0) k1), j0 = n3*8 + n4, k1 = 2kap (A), 2kap+1 (B), n2 = 0..7.
// Pure arithmetic (4 sincos + a packed power chain): the caller runs it ahead of the barrier that precedes p2_inv.
template <int LOGM>
__device__ __forceinline__ void p2_inv_twiddles(int t, C2 (&tw)[8]) {
    constexpr int M = Geo<LOGM>::M;
    const int kap = t >> 6, j0 = t & 63;
    const float2 ca = twiddle<M>(j0 * 2 * kap), cb = twiddle<M>(j0 * (2 * kap + 1));
    const float2 sa = twiddle<M / 128>(kap), sb = twiddle<M / 64>(2 * kap + 1);
    powers8(C2{pack(ca.x, cb.x), pack(ca.y, cb.y)}, C2{pack(sa.x, sb.x), pack(sa.y, sb.y)}, tw);
}
__device__ __forceinline__ void p2_inv(int t, float* re, float* im, const C2 (&tw)[8]) {
    const int kap = t >> 6, n3 = (t >> 3) & 7, n4 = t & 7;
    C2 v[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) v[r] = lds2(re, im, slot13(kap, brev<8>(r), n3, n4));
    dit8(v);
#pragma unroll
    for (int n2 = 0; n2 < 8; ++n2) sts2(re, im, slot13(kap, n2, n3, n4), cmul_conj(v[n2], tw[n2]));
}

// M = 4096: x[h*8 + n1] = unnormalised inverse at n = n1*512 + t + 256 h
__device__ __forceinline__ void p1_inv12(float2 (&x)[16], int t, const float* re, const float* im) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int j1 = t + 256 * h;
        const int n2 = j1 >> 6, n3 = (j1 >> 3) & 7, n4 = j1 & 7;
        C2 v[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) v[r] = lds2(re, im, slot13(brev<4>(r), n2, n3, n4));
        dit4(v);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            float2 s, d;
            unpack(v[i].r, s.x, d.x);
            unpack(v[i].i, s.y, d.y);
            switch (i) {      // d *= conj(w8^i)
                case 0: break;
                case 1: d = mul_w32<4, true>(d); break;
                case 2: d = mul_w32<8, true>(d); break;
                default: d = mul_w32<12, true>(d); break;
            }
            x[h * 8 + i] = amplfi::cadd(s, d);
            x[h * 8 + i + 4] = amplfi::csub(s, d);
        }
    }
}

// x[n1] = unnormalised inverse at n = n1*512 + t
__device__ __forceinline__ void p1_inv(float2 (&x)[16], int t, const float* re, const float* im) {
    const int n2 = t >> 6, n3 = (t >> 3) & 7, n4 = t & 7;
    C2 v[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) v[r] = lds2(re, im, slot13(brev<8>(r), n2, n3, n4));
    dit8(v);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        float2 s, d;
        unpack(v[i].r, s.x, d.x);
        unpack(v[i].i, s.y, d.y);
        switch (i) {      // d *= conj(w16^i)
            case 0: break;
            case 1: d = mul_w32<2, true>(d); break;
            case 2: d = mul_w32<4, true>(d); break;
            case 3: d = mul_w32<6, true>(d); break;
            case 4: d = mul_w32<8, true>(d); break;
            case 5: d = mul_w32<10, true>(d); break;
            case 6: d = mul_w32<12, true>(d); break;
            default: d = mul_w32<14, true>(d); break;
        }
        x[i] = amplfi::cadd(s, d);
        x[i + 8] = amplfi::csub(s, d);
    }
}

}  // namespace v2
}  // namespace amplfi
