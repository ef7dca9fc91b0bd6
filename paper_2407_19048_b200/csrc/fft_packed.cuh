// fft_packed.cuh -- packed-fp32x2 building blocks of the packed FFT passes (sm_100a; used through fft_tan.cuh).
//
// Blackwell issues add/mul/fma.f32x2 (SASS FADD2/FMUL2/FFMA2) on 64-bit register pairs: one issue slot for
// two fp32 lanes of work.  The FFT is bound by issue slots and the fp32 pipe (profiles/r02_ncu_inject_whiten.md), so the passes
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

}  // namespace pk
}  // namespace amplfi
