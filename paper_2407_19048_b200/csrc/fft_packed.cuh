// fft_packed.cuh -- packed-fp32x2 building blocks for the second-generation FFT passes (sm_100a).
//
// Blackwell issues add/mul/fma.f32x2 (SASS FADD2/FMUL2/FFMA2) on 64-bit register pairs: one issue slot for
// two fp32 lanes of work.  The FFT is issue-slot bound (profiles/r01_ncu_inject_whiten_v1.md), so the passes
// keep TWO butterflies per thread in a split layout: C2{r, i} with r = (re of butterfly A, re of butterfly B)
// and i = (im of A, im of B).  Complex add = 2 packed instructions for two complex adds, complex multiply =
// 4 for two; multiplication by +-i is a relabelling of r/i with a sign that folds into the next add.
#pragma once
#include <cuda_runtime.h>

#include "fft_core.cuh"

namespace amplfi {
namespace pk {

typedef unsigned long long u64;

__device__ __forceinline__ u64 pack(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unpack(u64 v, float& lo, float& hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
// negation written per half so that ptxas folds it into the consumer's operand modifier (-R.F32x2) instead of
// two LOP3 on the 64-bit pair
__device__ __forceinline__ u64 neg2(u64 a) { float lo, hi; unpack(a, lo, hi); return pack(-lo, -hi); }
__device__ __forceinline__ u64 bcast(float s) { return pack(s, s); }

struct C2 { u64 r, i; };          // two complex numbers: (A.re, B.re), (A.im, B.im)

__device__ __forceinline__ C2 cadd(C2 a, C2 b) { return C2{add2(a.r, b.r), add2(a.i, b.i)}; }
__device__ __forceinline__ C2 csub(C2 a, C2 b) { return C2{sub2(a.r, b.r), sub2(a.i, b.i)}; }
// a * w (element-wise on both halves)
__device__ __forceinline__ C2 cmul(C2 a, C2 w) {
    u64 t = mul2(a.i, w.i);
    u64 u = mul2(a.i, w.r);
    return C2{fma2(a.r, w.r, neg2(t)), fma2(a.r, w.i, u)};
}
// a * conj(w)
__device__ __forceinline__ C2 cmul_conj(C2 a, C2 w) {
    u64 t = mul2(a.i, w.i);
    u64 u = mul2(a.r, w.i);
    return C2{fma2(a.r, w.r, t), fma2(a.i, w.r, neg2(u))};
}
// both halves times the same scalar complex w / conj(w)
__device__ __forceinline__ C2 cmul_s(C2 a, float2 w) { return cmul(a, C2{bcast(w.x), bcast(w.y)}); }
__device__ __forceinline__ C2 cmul_conj_s(C2 a, float2 w) { return cmul_conj(a, C2{bcast(w.x), bcast(w.y)}); }
__device__ __forceinline__ C2 mul_negi(C2 a) { return C2{a.i, neg2(a.r)}; }   // * (-i)
__device__ __forceinline__ C2 mul_posi(C2 a) { return C2{neg2(a.i), a.r}; }   // * (+i)

constexpr float kH = 0.70710678118654752f;

// a * exp(-2 pi i j / 8) (INV: conjugate), j compile-time in [0, 4)
template <int J, bool INV>
__device__ __forceinline__ C2 mul_w8(C2 a) {
    if constexpr (J == 0) {
        return a;
    } else if constexpr (J == 2) {
        return INV ? mul_posi(a) : mul_negi(a);
    } else if constexpr (J == 1) {
        const u64 h = bcast(kH);
        // fwd (1 - i)/sqrt2: (re + im, im - re) h ; inv (1 + i)/sqrt2: (re - im, re + im) h
        return INV ? C2{mul2(sub2(a.r, a.i), h), mul2(add2(a.r, a.i), h)}
                   : C2{mul2(add2(a.r, a.i), h), mul2(sub2(a.i, a.r), h)};
    } else {
        const u64 h = bcast(kH), nh = bcast(-kH);
        // fwd (-1 - i)/sqrt2: (im - re, -(re + im)) h ; inv (-1 + i)/sqrt2: (-(re + im), re - im) h
        return INV ? C2{mul2(add2(a.r, a.i), nh), mul2(sub2(a.r, a.i), h)}
                   : C2{mul2(sub2(a.i, a.r), h), mul2(add2(a.r, a.i), nh)};
    }
}

// Forward DFT_8 on both halves: natural-order input, output q left in v[brev<8>(q)].
__device__ __forceinline__ void dif8(C2 (&v)[8]) {
    C2 d;
#define AMPLFI_BF(i, j, TW) d = csub(v[i], v[j]); v[i] = cadd(v[i], v[j]); v[j] = TW;
    AMPLFI_BF(0, 4, d) AMPLFI_BF(1, 5, (mul_w8<1, false>(d))) AMPLFI_BF(2, 6, (mul_w8<2, false>(d))) AMPLFI_BF(3, 7, (mul_w8<3, false>(d)))
    AMPLFI_BF(0, 2, d) AMPLFI_BF(1, 3, (mul_w8<2, false>(d))) AMPLFI_BF(4, 6, d) AMPLFI_BF(5, 7, (mul_w8<2, false>(d)))
    AMPLFI_BF(0, 1, d) AMPLFI_BF(2, 3, d) AMPLFI_BF(4, 5, d) AMPLFI_BF(6, 7, d)
#undef AMPLFI_BF
}
// Unnormalised inverse DFT_8 on both halves: input q taken from v[brev<8>(q)], natural-order output.
__device__ __forceinline__ void dit8(C2 (&v)[8]) {
    C2 b;
#define AMPLFI_BT(i, j, TW) b = TW; v[j] = csub(v[i], b); v[i] = cadd(v[i], b);
    AMPLFI_BT(0, 1, v[1]) AMPLFI_BT(2, 3, v[3]) AMPLFI_BT(4, 5, v[5]) AMPLFI_BT(6, 7, v[7])
    AMPLFI_BT(0, 2, v[2]) AMPLFI_BT(1, 3, (mul_w8<2, true>(v[3]))) AMPLFI_BT(4, 6, v[6]) AMPLFI_BT(5, 7, (mul_w8<2, true>(v[7])))
    AMPLFI_BT(0, 4, v[4]) AMPLFI_BT(1, 5, (mul_w8<1, true>(v[5]))) AMPLFI_BT(2, 6, (mul_w8<2, true>(v[6]))) AMPLFI_BT(3, 7, (mul_w8<3, true>(v[7])))
#undef AMPLFI_BT
}

// scalar complex helpers for twiddle chains
__device__ __forceinline__ float2 csq(float2 a) { return make_float2(a.x * a.x - a.y * a.y, 2.0f * a.x * a.y); }

// g[q] = base * step^q, q = 0..7 (scalar chain; depth 3)
__device__ __forceinline__ void powers8(float2 base, float2 step, float2 (&g)[8]) {
    const float2 s2 = csq(step), s4 = csq(s2);
    g[0] = base;
    g[1] = amplfi::cmul(base, step);
    g[2] = amplfi::cmul(g[0], s2);
    g[3] = amplfi::cmul(g[1], s2);
    g[4] = amplfi::cmul(g[0], s4);
    g[5] = amplfi::cmul(g[1], s4);
    g[6] = amplfi::cmul(g[2], s4);
    g[7] = amplfi::cmul(g[3], s4);
}
// packed version: G[q] = BASE * STEP^q on both halves independently
__device__ __forceinline__ void powers8(C2 base, C2 step, C2 (&g)[8]) {
    const C2 s2 = cmul(step, step), s4 = cmul(s2, s2);
    g[0] = base;
    g[1] = cmul(base, step);
    g[2] = cmul(g[0], s2);
    g[3] = cmul(g[1], s2);
    g[4] = cmul(g[0], s4);
    g[5] = cmul(g[1], s4);
    g[6] = cmul(g[2], s4);
    g[7] = cmul(g[3], s4);
}

}  // namespace pk
}  // namespace amplfi
