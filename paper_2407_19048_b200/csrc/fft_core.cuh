// fft_core.cuh -- register/shared-memory complex FFT building blocks for sm_100a.
//
// A real segment of N = 2M samples is packed as M complex points z[m] = x[2m] + i x[2m+1] and
// transformed by a three-pass in-place decimation-in-frequency FFT, M = RA * RB * RC:
//   pass A  butterflies over the most significant input digit, operands straight from global memory,
//   pass B  over the middle digit (shared memory in, shared memory out),
//   pass C  over the least significant digit; its outputs stay in REGISTERS.
// Each thread of pass C owns the two butterflies that hold bins {k} and {M - k}, so the real-FFT
// split, the per-bin work (injection, whitening, |X|^2 ...) and the merge for the inverse transform
// need no further exchange.  The inverse runs the same passes backwards (C', B', A') as a
// decimation-in-time FFT and stores natural-order time samples to global memory.
// Forward kernel exp(-2 pi i k n / M); the inverse is unnormalised (callers fold 1/M into a scale).
//
// Shared-memory layout: position p = kA * LB + kB * RC + kC (LB = RB * RC), physical slot
// p ^ ((p >> log2 LB) & 15): the XOR with the low bits of kA makes the stride-LB accesses of pass C
// bank-conflict free while leaving the unit-stride accesses of passes A and B conflict free.
#pragma once
#include <cuda_runtime.h>

namespace amplfi {

// cos/sin of 2 pi m / 32, m = 0..15
__device__ constexpr float kCos32[16] = {
    1.0f, 0.98078528040323044f, 0.92387953251128674f, 0.83146961230254524f,
    0.70710678118654752f, 0.55557023301960222f, 0.38268343236508977f, 0.19509032201612827f,
    0.0f, -0.19509032201612827f, -0.38268343236508977f, -0.55557023301960222f,
    -0.70710678118654752f, -0.83146961230254524f, -0.92387953251128674f, -0.98078528040323044f};
__device__ constexpr float kSin32[16] = {
    0.0f, 0.19509032201612827f, 0.38268343236508977f, 0.55557023301960222f,
    0.70710678118654752f, 0.83146961230254524f, 0.92387953251128674f, 0.98078528040323044f,
    1.0f, 0.98078528040323044f, 0.92387953251128674f, 0.83146961230254524f,
    0.70710678118654752f, 0.55557023301960222f, 0.38268343236508977f, 0.19509032201612827f};

__host__ __device__ constexpr int ilog2(int x) { return x <= 1 ? 0 : 1 + ilog2(x >> 1); }

template <int R>
__host__ __device__ constexpr int brev(int i) {
    int r = 0;
    for (int b = 0; b < ilog2(R); ++b) r |= ((i >> b) & 1) << (ilog2(R) - 1 - b);
    return r;
}

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    return make_float2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x);
}
__device__ __forceinline__ float2 cmul_conj(float2 a, float2 w) {   // a * conj(w)
    return make_float2(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y);
}
__device__ __forceinline__ float2 cconj(float2 a) { return make_float2(a.x, -a.y); }

// a * exp(-+ 2 pi i m / 32) with m a compile-time constant in [0, 16); INV selects the + sign.
template <int M32, bool INV>
__device__ __forceinline__ float2 mul_w32(float2 a) {
    if constexpr (M32 == 0) {
        return a;
    } else if constexpr (M32 == 8) {          // -i (forward) or +i (inverse)
        return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
    } else if constexpr (M32 == 4) {          // (1 -+ i)/sqrt2
        constexpr float h = 0.70710678118654752f;
        return INV ? make_float2((a.x - a.y) * h, (a.x + a.y) * h) : make_float2((a.x + a.y) * h, (a.y - a.x) * h);
    } else if constexpr (M32 == 12) {         // (-1 -+ i)/sqrt2
        constexpr float h = 0.70710678118654752f;
        return INV ? make_float2((-a.x - a.y) * h, (a.x - a.y) * h) : make_float2((a.y - a.x) * h, (-a.x - a.y) * h);
    } else {
        constexpr float c = kCos32[M32];
        constexpr float s = INV ? kSin32[M32] : -kSin32[M32];
        return make_float2(a.x * c - a.y * s, a.x * s + a.y * c);
    }
}

template <int R, int S, int I, bool INV>
struct StageStep {
    // one radix-2 butterfly of the stage with half-size S acting on v[I], v[I+S]
    static __device__ __forceinline__ void dif(float2 (&v)[R]) {
        if constexpr ((I & S) == 0) {
            float2 a = v[I], b = v[I + S];
            v[I] = cadd(a, b);
            v[I + S] = mul_w32<(I & (S - 1)) * (16 / S), INV>(csub(a, b));
        }
    }
    static __device__ __forceinline__ void dit(float2 (&v)[R]) {
        if constexpr ((I & S) == 0) {
            float2 a = v[I], b = mul_w32<(I & (S - 1)) * (16 / S), INV>(v[I + S]);
            v[I] = cadd(a, b);
            v[I + S] = csub(a, b);
        }
    }
};

template <int R, int S, bool INV, int I = 0>
__device__ __forceinline__ void stage_dif(float2 (&v)[R]) {
    if constexpr (I < R) {
        StageStep<R, S, I, INV>::dif(v);
        stage_dif<R, S, INV, I + 1>(v);
    }
}
template <int R, int S, bool INV, int I = 0>
__device__ __forceinline__ void stage_dit(float2 (&v)[R]) {
    if constexpr (I < R) {
        StageStep<R, S, I, INV>::dit(v);
        stage_dit<R, S, INV, I + 1>(v);
    }
}

// Forward DFT_R of v (kernel e^{-i}): natural-order input, output k is left in v[brev<R>(k)].
template <int R, int S = R / 2>
__device__ __forceinline__ void fft_dif_fwd(float2 (&v)[R]) {
    if constexpr (S >= 1) {
        stage_dif<R, S, false>(v);
        fft_dif_fwd<R, S / 2>(v);
    }
}
// Unnormalised inverse DFT_R (kernel e^{+i}): input k taken from v[brev<R>(k)], natural-order output.
template <int R, int S = 1>
__device__ __forceinline__ void fft_dit_inv(float2 (&v)[R]) {
    if constexpr (S < R) {
        stage_dit<R, S, true>(v);
        fft_dit_inv<R, S * 2>(v);
    }
}

// exp(-2 pi i m / L) for an integer m in [0, L): argument reduced to [-pi, pi] before the fast
// sine/cosine (absolute error ~4e-7).
template <int L>
__device__ __forceinline__ float2 twiddle(int m) {
    m &= (L - 1);
    if (m >= L / 2) m -= L;
    float ang = (float)m * (-6.283185307179586f / (float)L);
    float s, c;
    __sincosf(ang, &s, &c);
    return make_float2(c, s);
}

// ------------------------------------------------------------------------------------------------
// Plan of the three-pass transform for M = 2^LOGM complex points.
// E elements per thread, RC = E/2 (one {k, M-k} butterfly pair per thread), T = RA*RB/2 threads.
// ------------------------------------------------------------------------------------------------
template <int LOGM> struct FftPlan;
template <> struct FftPlan<14> { static constexpr int RA = 32, RB = 32, RC = 16; };
template <> struct FftPlan<13> { static constexpr int RA = 32, RB = 16, RC = 16; };
template <> struct FftPlan<12> { static constexpr int RA = 16, RB = 16, RC = 16; };
template <> struct FftPlan<11> { static constexpr int RA = 16, RB = 8,  RC = 16; };
template <> struct FftPlan<10> { static constexpr int RA = 16, RB = 8,  RC = 8;  };
template <> struct FftPlan<9>  { static constexpr int RA = 8,  RB = 8,  RC = 8;  };

template <int LOGM>
struct Fft {
    using P = FftPlan<LOGM>;
    static constexpr int M = 1 << LOGM;
    static constexpr int RA = P::RA, RB = P::RB, RC = P::RC;
    static constexpr int E = 2 * RC;
    static constexpr int T = RA * RB / 2;            // threads per CTA
    static constexpr int LB = RB * RC;               // length of a pass-B block
    static constexpr int LOGLB = ilog2(LB);
    static constexpr int NA = E / RA;                // butterflies per thread in pass A
    static constexpr int NB = E / RB;                // ... in pass B
    static constexpr size_t SMEM_BYTES = (size_t)M * sizeof(float2);
    static_assert(RA * RB * RC == M && NA >= 1 && NB >= 1, "bad plan");

    static __device__ __forceinline__ int phys(int p) { return p ^ ((p >> LOGLB) & 15); }

    // ---- pass A forward: v[nA] = z[nA*LB + jA] already loaded; butterfly, twiddle, store to smem ----
    static __device__ __forceinline__ void pass_a_fwd(float2 (&v)[RA], int jA, float2* sm) {
        fft_dif_fwd<RA>(v);
#pragma unroll
        for (int i = 0; i < RA; ++i) {
            const int kA = brev<RA>(i);
            float2 val = v[i];
            if (kA != 0) val = cmul(val, twiddle<M>(jA * kA));
            sm[phys(kA * LB + jA)] = val;
        }
    }
    // ---- pass B forward: butterfly g -> (kA, nC); in place ----
    static __device__ __forceinline__ void pass_b_fwd(int g, float2* sm) {
        const int nC = g & (RC - 1);
        const int kA = g / RC;
        float2 v[RB];
#pragma unroll
        for (int nB = 0; nB < RB; ++nB) v[nB] = sm[phys(kA * LB + nB * RC + nC)];
        fft_dif_fwd<RB>(v);
#pragma unroll
        for (int i = 0; i < RB; ++i) {
            const int kB = brev<RB>(i);
            float2 val = v[i];
            if (kB != 0) val = cmul(val, twiddle<LB>(nC * kB));
            sm[phys(kA * LB + kB * RC + nC)] = val;
        }
    }
    // ---- pass C forward: butterfly with low frequency part klow = kA + RA*kB; output kC in v[brev(kC)] ----
    static __device__ __forceinline__ void pass_c_fwd(int klow, float2 (&v)[RC], const float2* sm) {
        const int kA = klow & (RA - 1);
        const int kB = klow / RA;
        const int base = kA * LB + kB * RC;
#pragma unroll
        for (int nC = 0; nC < RC; ++nC) v[nC] = sm[phys(base + nC)];
        fft_dif_fwd<RC>(v);
    }
    // ---- pass C inverse: v[brev(kC)] -> time digit nC, conj twiddle of pass B, store ----
    static __device__ __forceinline__ void pass_c_inv(int klow, float2 (&v)[RC], float2* sm) {
        const int kA = klow & (RA - 1);
        const int kB = klow / RA;
        const int base = kA * LB + kB * RC;
        fft_dit_inv<RC>(v);
#pragma unroll
        for (int nC = 0; nC < RC; ++nC) {
            float2 val = v[nC];
            if (nC != 0) val = cmul_conj(val, twiddle<LB>(nC * kB));
            sm[phys(base + nC)] = val;
        }
    }
    // ---- pass B inverse ----
    static __device__ __forceinline__ void pass_b_inv(int g, float2* sm) {
        const int nC = g & (RC - 1);
        const int kA = g / RC;
        float2 v[RB];
#pragma unroll
        for (int i = 0; i < RB; ++i) v[i] = sm[phys(kA * LB + brev<RB>(i) * RC + nC)];
        fft_dit_inv<RB>(v);
#pragma unroll
        for (int nB = 0; nB < RB; ++nB) {
            float2 val = v[nB];
            const int jA = nB * RC + nC;
            val = cmul_conj(val, twiddle<M>(jA * kA));
            sm[phys(kA * LB + jA)] = val;
        }
    }
    // ---- pass A inverse: gather kA digits, butterfly; v[nA] = z'[nA*LB + jA] (unnormalised) ----
    static __device__ __forceinline__ void pass_a_inv(float2 (&v)[RA], int jA, const float2* sm) {
#pragma unroll
        for (int i = 0; i < RA; ++i) v[i] = sm[phys(brev<RA>(i) * LB + jA)];
        fft_dit_inv<RA>(v);
    }
};

// Real-FFT split for the bin pair (k, M-k), 0 < k < M/2 or k = M/2 (then zb == za):
// given za = Z[k], zb = Z[M-k] returns 2*X[k] and 2*X[M-k] of the length-2M real transform,
// w = exp(-2 pi i k / (2M)).
__device__ __forceinline__ void split_pair(float2 za, float2 zb, float2 w, float2& xa2, float2& xb2) {
    float2 e = make_float2(za.x + zb.x, za.y - zb.y);            // za + conj(zb)       = 2E
    float2 d = make_float2(za.x - zb.x, za.y + zb.y);            // za - conj(zb)
    float2 o = make_float2(d.y, -d.x);                           // -i * d              = 2O
    float2 wo = cmul(o, w);
    xa2 = cadd(e, wo);                                           // 2X[k]   = 2E + w^k 2O
    float2 t = csub(e, wo);
    xb2 = cconj(t);                                              // 2X[M-k] = conj(2E - w^k 2O)
}
// Inverse of split_pair up to a factor: given Ya = Y[k], Yb = Y[M-k] returns 2*Z'[k], 2*Z'[M-k]
// with Z' = E' + i O', E' = (Ya + conj Yb)/2, O' = conj(w) (Ya - conj Yb)/2.
__device__ __forceinline__ void merge_pair(float2 ya, float2 yb, float2 w, float2& za2, float2& zb2) {
    float2 e = make_float2(ya.x + yb.x, ya.y - yb.y);            // 2E'
    float2 d = make_float2(ya.x - yb.x, ya.y + yb.y);
    float2 o = cmul_conj(d, w);                                  // 2O'
    za2 = make_float2(e.x - o.y, e.y + o.x);                     // 2E' + i 2O'
    zb2 = make_float2(e.x + o.y, o.x - e.y);                     // conj(2E') + i conj(2O')
}

// Visit every bin held by a pass-C thread.  Thread `tid` (0 <= tid < T) holds butterflies
// klow_a = tid and klow_b = RA*RB - tid (tid > 0), or klow_a = 0 and klow_b = RA*RB/2 (tid == 0); load them
// with pass_c_klow().  fpair(k, za, zb) is called with za = Z[k], zb = Z[M-k] (by reference, 0 < k < M/2);
// fself(k, z) for k = M/2 and fdc(z) for Z[0] (which carries the DC and Nyquist bins of the real transform).
template <int LOGM>
__device__ __forceinline__ void pass_c_klow(int tid, int& klow_a, int& klow_b) {
    using F = Fft<LOGM>;
    klow_a = tid;
    klow_b = (tid == 0) ? (F::RA * F::RB / 2) : (F::RA * F::RB - tid);
}

template <int LOGM, class FPair, class FSelf, class FDc>
__device__ __forceinline__ void for_each_bin_pair(int tid, float2 (&va)[Fft<LOGM>::RC], float2 (&vb)[Fft<LOGM>::RC],
                                                  FPair fpair, FSelf fself, FDc fdc) {
    using F = Fft<LOGM>;
    constexpr int RC = F::RC, RAB = F::RA * F::RB;
    if (tid != 0) {
#pragma unroll
        for (int i = 0; i < RC; ++i) fpair(tid + RAB * brev<RC>(i), va[i], vb[RC - 1 - i]);
    } else {
        fdc(va[0]);
        fself(RAB * (RC / 2), va[brev<RC>(RC / 2)]);
#pragma unroll
        for (int q = 1; q < RC / 2; ++q) fpair(RAB * q, va[brev<RC>(q)], va[brev<RC>(RC - q)]);
#pragma unroll
        for (int q = 0; q < RC / 2; ++q) fpair(RAB / 2 + RAB * q, vb[brev<RC>(q)], vb[brev<RC>(RC - 1 - q)]);
    }
}

}  // namespace amplfi
