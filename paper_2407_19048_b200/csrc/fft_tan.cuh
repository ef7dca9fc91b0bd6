// fft_tan.cuh -- radix-2 decimation-in-time butterflies with the twiddle in "cosine-tangent" form, packed fp32x2.
//
// A DIT butterfly with twiddle T = c (1 + i tau)  (c = Re T, tau = Im T / Re T) is
//     u = b.re - tau b.im,  v = b.im + tau b.re,    a' = a + c (u + i v),    b' = a - c (u + i v)
// i.e. SIX fused multiply-adds instead of the 4 (complex multiply) + 4 (add/sub) of the textbook form.  A radix-16 pass
// whose inputs carry the inter-pass twiddle W^r (W = per-thread constant) is the same radix-2 network with the twiddles
//     level 2:  W^8      level 4:  W^4 (x -i)      level 8:  W^2, W^2 w8 (x -i)      level 16:  W w16^q, q < 4 (x -i)
// so the inter-pass twiddle costs nothing extra: 32 butterflies x 6 FMA = 12 lane-operations per point and pass against
// 14.25 for butterflies with exact constants followed by a twiddle multiplication.  Multiplication of T by -i (forward) /
// +i (inverse) is a relabelling of (u, v).  |c| is kept away from zero by the producers of (c, tau) (tables: fp64, clamped;
// on the fly: c + 1e-8), the rounding error of c * (tau * x) is that of Im T * x.
//
// Lanes: C2{r, i} holds two complex numbers (A.re, B.re), (A.im, B.im) (fft_packed.cuh); a twiddle is either per lane
// (Tw2: packed c, packed tau) or shared (Tw1: scalars, broadcast by the FFMA2 operand modifier R.F32).
#pragma once
#include "fft_packed.cuh"

namespace amplfi {
namespace tn {

using namespace pk;

struct Tw2 { u64 c, t; };          // per-lane twiddle: (cA, cB), (tauA, tauB)
struct Tw1 { float c, t; };        // the same twiddle for both lanes

__device__ __forceinline__ u64 bc(float s) { return pack(s, s); }     // folds into the .F32 operand form of FFMA2

// a <- a + T b, b <- a - T b with T = c (1 + i tau) [INV: conj T], ROT: T times -i [INV: +i];
// CONJB: the second output is left conjugated (its imaginary part negated through the operand modifiers, no extra work)
template <bool INV, bool ROT, bool CONJB = false>
__device__ __forceinline__ void bf(C2& a, C2& b, u64 c, u64 t) {
    const u64 u = INV ? fma2(t, b.i, b.r) : fma2(neg2(t), b.i, b.r);
    const u64 v = INV ? fma2(neg2(t), b.r, b.i) : fma2(t, b.r, b.i);
    const C2 a0 = a;
    const u64 nc = neg2(c), nai = neg2(a0.i);
    if (!ROT) {
        a.r = fma2(c, u, a0.r);   a.i = fma2(c, v, a0.i);
        b.r = fma2(nc, u, a0.r);  b.i = CONJB ? fma2(c, v, nai) : fma2(nc, v, a0.i);
    } else if (!INV) {                 // -i (u + i v) = v - i u
        a.r = fma2(c, v, a0.r);   a.i = fma2(nc, u, a0.i);
        b.r = fma2(nc, v, a0.r);  b.i = CONJB ? fma2(nc, u, nai) : fma2(c, u, a0.i);
    } else {                           // +i (u + i v) = -v + i u
        a.r = fma2(nc, v, a0.r);  a.i = fma2(c, u, a0.i);
        b.r = fma2(c, v, a0.r);   b.i = CONJB ? fma2(c, u, nai) : fma2(nc, u, a0.i);
    }
}
template <bool INV, bool ROT, bool CONJB = false> __device__ __forceinline__ void bf(C2& a, C2& b, Tw2 w) { bf<INV, ROT, CONJB>(a, b, w.c, w.t); }
template <bool INV, bool ROT, bool CONJB = false> __device__ __forceinline__ void bf(C2& a, C2& b, Tw1 w) { bf<INV, ROT, CONJB>(a, b, bc(w.c), bc(w.t)); }

// T = 1 (ROT: -i forward, +i inverse): four additions
template <bool INV, bool ROT>
__device__ __forceinline__ void bf1(C2& a, C2& b) {
    const C2 a0 = a, b0 = b;
    if (!ROT) {
        a = cadd(a0, b0); b = csub(a0, b0);
    } else if (!INV) {                 // -i b = (b.i, -b.r)
        a.r = add2(a0.r, b0.i); a.i = sub2(a0.i, b0.r);
        b.r = sub2(a0.r, b0.i); b.i = add2(a0.i, b0.r);
    } else {                           // +i b = (-b.i, b.r)
        a.r = sub2(a0.r, b0.i); a.i = add2(a0.i, b0.r);
        b.r = add2(a0.r, b0.i); b.i = sub2(a0.i, b0.r);
    }
}
// T = w8 = (1 - i)/sqrt2 (INV: conj): tau = -1 (INV: applied with the conjugate formulas), c = 1/sqrt2
template <bool INV, bool ROT>
__device__ __forceinline__ void bf_w8(C2& a, C2& b) {
    const u64 u = INV ? sub2(b.r, b.i) : add2(b.r, b.i);      // fwd: b.r - tau b.i = b.r + b.i; inv: b.r + tau b.i
    const u64 v = INV ? add2(b.i, b.r) : sub2(b.i, b.r);
    const u64 c = bc(kH);
    const C2 a0 = a;
    if (!ROT) {
        a.r = fma2(c, u, a0.r);        a.i = fma2(c, v, a0.i);
        b.r = fma2(neg2(c), u, a0.r);  b.i = fma2(neg2(c), v, a0.i);
    } else if (!INV) {
        a.r = fma2(c, v, a0.r);        a.i = fma2(neg2(c), u, a0.i);
        b.r = fma2(neg2(c), v, a0.r);  b.i = fma2(c, u, a0.i);
    } else {
        a.r = fma2(neg2(c), v, a0.r);  a.i = fma2(c, u, a0.i);
        b.r = fma2(c, v, a0.r);        b.i = fma2(neg2(c), u, a0.i);
    }
}

// exact constants of w16 = exp(-2 pi i / 16) and w16^3 in (c, tau) form
constexpr float kC16_1 = 0.92387953251128674f, kT16_1 = -0.41421356237309505f;     // cos(pi/8), -tan(pi/8)
constexpr float kC16_3 = 0.38268343236508977f, kT16_3 = -2.4142135623730950f;      // cos(3pi/8), -tan(3pi/8)

// X[q] = sum_r y[r] W^r w16^(rq) (INV: conjugate kernel), y[r] taken from v[brev16(r)], X[q] left in v[q].
//   tw[0] = W^8, tw[1] = W^4, tw[2] = W^2, tw[3] = W^2 w8, tw[4 + q] = W w16^q (q < 4)   (forward-sign twiddles)
// CONJ_HI: outputs X[8..15] are left conjugated
template <bool INV, class TW, bool CONJ_HI = false>
__device__ __forceinline__ void dit16(C2 (&v)[16], const TW (&tw)[8]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) bf<INV, false>(v[2 * i], v[2 * i + 1], tw[0]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        bf<INV, false>(v[4 * i], v[4 * i + 2], tw[1]);
        bf<INV, true>(v[4 * i + 1], v[4 * i + 3], tw[1]);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        bf<INV, false>(v[8 * i], v[8 * i + 4], tw[2]);
        bf<INV, false>(v[8 * i + 1], v[8 * i + 5], tw[3]);
        bf<INV, true>(v[8 * i + 2], v[8 * i + 6], tw[2]);
        bf<INV, true>(v[8 * i + 3], v[8 * i + 7], tw[3]);
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        bf<INV, false, CONJ_HI>(v[q], v[q + 8], tw[4 + q]);
        bf<INV, true, CONJ_HI>(v[q + 4], v[q + 12], tw[4 + q]);
    }
}

// the same with W = 1: exact constants, trivial butterflies as additions
template <bool INV>
__device__ __forceinline__ void dit16_const(C2 (&v)[16]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) bf1<INV, false>(v[2 * i], v[2 * i + 1]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        bf1<INV, false>(v[4 * i], v[4 * i + 2]);
        bf1<INV, true>(v[4 * i + 1], v[4 * i + 3]);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        bf1<INV, false>(v[8 * i], v[8 * i + 4]);
        bf_w8<INV, false>(v[8 * i + 1], v[8 * i + 5]);
        bf1<INV, true>(v[8 * i + 2], v[8 * i + 6]);
        bf_w8<INV, true>(v[8 * i + 3], v[8 * i + 7]);
    }
    bf1<INV, false>(v[0], v[8]);
    bf<INV, false>(v[1], v[9], Tw1{kC16_1, kT16_1});
    bf_w8<INV, false>(v[2], v[10]);
    bf<INV, false>(v[3], v[11], Tw1{kC16_3, kT16_3});
    bf1<INV, true>(v[4], v[12]);
    bf<INV, true>(v[5], v[13], Tw1{kC16_1, kT16_1});
    bf_w8<INV, true>(v[6], v[14]);
    bf<INV, true>(v[7], v[15], Tw1{kC16_3, kT16_3});
}

// radix 8 (W general): tw[0] = W^4, tw[1] = W^2, tw[2 + q] = W w8^q (q < 2); y[r] from v[brev8(r)];
// CONJ_HI: outputs X[4..7] are left conjugated
template <bool INV, class TW, bool CONJ_HI = false>
__device__ __forceinline__ void dit8(C2 (&v)[8], const TW (&tw)[8]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) bf<INV, false>(v[2 * i], v[2 * i + 1], tw[0]);
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        bf<INV, false>(v[4 * i], v[4 * i + 2], tw[1]);
        bf<INV, true>(v[4 * i + 1], v[4 * i + 3], tw[1]);
    }
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        bf<INV, false, CONJ_HI>(v[q], v[q + 4], tw[2 + q]);
        bf<INV, true, CONJ_HI>(v[q + 2], v[q + 6], tw[2 + q]);
    }
}
// radix 4: tw[0] = W^2, tw[1] = W; y[r] from v[brev4(r)];  CONJ_HI: outputs X[2], X[3] are left conjugated
template <bool INV, class TW, bool CONJ_HI = false>
__device__ __forceinline__ void dit4(C2 (&v)[4], const TW (&tw)[8]) {
    bf<INV, false>(v[0], v[1], tw[0]);
    bf<INV, false>(v[2], v[3], tw[0]);
    bf<INV, false, CONJ_HI>(v[0], v[2], tw[1]);
    bf<INV, true, CONJ_HI>(v[1], v[3], tw[1]);
}
// radix R in {4, 8, 16} with the twiddle row layout of each (entries beyond the radix's need are unused)
template <int R, bool INV, class TW, bool CONJ_HI = false>
__device__ __forceinline__ void dit_r(C2 (&v)[R], const TW (&tw)[8]) {
    if constexpr (R == 16) dit16<INV, TW, CONJ_HI>(v, tw);
    else if constexpr (R == 8) dit8<INV, TW, CONJ_HI>(v, tw);
    else dit4<INV, TW, CONJ_HI>(v, tw);
}

// (c, tau) of exp(i theta) computed on the fly: theta in [-pi, pi]; c is nudged off an exact zero by 1e-8 (below half an ulp
// of every |c| > 0.25; nearer to a zero of the cosine c * tau still equals the computed sine and the c * x term moves by
// 1e-8 |x|, under fp32 rounding of the result; tau stays below ~1e8 so that large spectra (filter design) cannot overflow)
__device__ __forceinline__ Tw1 tan_twiddle(float theta) {
    float s, c;
    __sincosf(theta, &s, &c);
    c += 1e-8f;
    return Tw1{c, __fdividef(s, c)};
}

// scalar butterfly of the same form on float2 values: lo <- a + T b, hi <- a - T b
template <bool INV, bool ROT>
__device__ __forceinline__ void bf_s(float2 a, float2 b, Tw1 w, float2& lo, float2& hi) {
    const float u = INV ? fmaf(w.t, b.y, b.x) : fmaf(-w.t, b.y, b.x);
    const float v = INV ? fmaf(-w.t, b.x, b.y) : fmaf(w.t, b.x, b.y);
    float pr, pi;
    if (!ROT) { pr = u; pi = v; }
    else if (!INV) { pr = v; pi = -u; }
    else { pr = -v; pi = u; }
    lo = make_float2(fmaf(w.c, pr, a.x), fmaf(w.c, pi, a.y));
    hi = make_float2(fmaf(-w.c, pr, a.x), fmaf(-w.c, pi, a.y));
}

}  // namespace tn
}  // namespace amplfi
