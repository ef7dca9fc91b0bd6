// inject_whiten13.cu -- fused gather -> FFT -> inject -> whiten -> iFFT for n = 16384 (configs c1, c2, c3),
// second generation: 4 passes (16*8*8*8), 16 points per thread, 512 threads per segment, packed fp32x2 math,
// 2 CTAs (32 warps) per SM.  See inject_whiten_v2.cuh for the index algebra.  PAPER.md:103, :105.
#include "amplfi_internal.h"
#include "inject_whiten_v2.cuh"

namespace amplfi {

using namespace v2;

// VT virtual threads (of the 512 the index algebra is written for) per physical thread: VT = 2 runs 256 threads with
// 128 registers, trading thread-level for instruction-level parallelism (loads of one virtual thread overlap the
// arithmetic of the other).
// VIEWS = 2 (MODE_FUSED only): the two data views d, d' of PAPER.md:93, :117 from ONE forward transform.  The forward
// spectrum of every virtual thread is parked in the second view's own output row (64 KB, exactly the row size; it stays
// in L2 until that view's samples overwrite it) and read back for the second pointwise stage + inverse transform.
template <int LOGM, int MODE, int VT, bool FWD, int VIEWS>
__global__ void __launch_bounds__(Geo<LOGM>::T / VT, LOGM == 13 ? 2 : (LOGM == 12 ? 4 : 8)) inject_whiten13_kernel(const IwArgs a, int units) {
    using G = Geo<LOGM>;
    constexpr int TT = G::T / VT;
    constexpr int M = G::M, N = G::N, K = G::M + 1, KL = G::KL;
    extern __shared__ float smem13[];
    float* re = smem13;
    float* im = smem13 + M;
    const int unit = blockIdx.x, tt = threadIdx.x;
    const int b = unit / a.n_det, d = unit - b * a.n_det;

    // ---- a-5 gather ----
    const float* x = nullptr;
    const int n_out = N - 2 * a.crop;
    float* out = a.out + (size_t)unit * n_out;
    constexpr bool fwd = FWD;                              // false: inverse-only launch, the spectrum starts at zero
    if (!fwd) {
    } else if (a.offsets != nullptr) {
        const long off = a.offsets[unit];
        if (off < 0 || off + N > a.strip_len) {            // never read out of bounds: poison the row instead
            const float qnan = __int_as_float(0x7fc00000);
            for (int i = tt; i < n_out; i += TT) out[i] = qnan;
            if constexpr (VIEWS == 2) {                      // the second view's row as well
                float* o2 = a.out2 + (size_t)unit * N;
                for (int i = tt; i < N; i += TT) o2[i] = qnan;
            }
            return;
        }
        x = a.noise + (size_t)d * a.strip_len + off;
    } else {
        x = a.noise + (size_t)unit * N;
    }

    // L2 prefetch of the segment a CTA one wave later will gather (one bulk instruction for the whole 64 KB):
    // the head-of-CTA loads then hit L2 instead of waiting on HBM.
    if (tt == 0 && fwd) {
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
            if (ok) {
                const size_t p0 = (reinterpret_cast<size_t>(nx) + 15) & ~(size_t)15;      // inside the segment
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p0), "r"(N * 4 - 16) : "memory");
            }
        }
    }

    // ---- a-6 forward real FFT of the packed sequence z[m] = x[2m] + i x[2m+1] ----
    if (fwd) {
        float2 z[VT][16];
        if ((reinterpret_cast<size_t>(x) & 7) == 0) {
            const float2* x2 = reinterpret_cast<const float2*>(x);
#pragma unroll
            for (int vt = 0; vt < VT; ++vt)
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1) z[vt][n1] = __ldcs(x2 + sample_index<LOGM>(n1, tt + vt * TT));
        } else {
#pragma unroll
            for (int vt = 0; vt < VT; ++vt)
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1) {
                    const int m = sample_index<LOGM>(n1, tt + vt * TT);
                    z[vt][n1] = make_float2(__ldg(x + 2 * m), __ldg(x + 2 * m + 1));
                }
        }
#pragma unroll
        for (int vt = 0; vt < VT; ++vt) {
            if constexpr (LOGM == 13) p1_fwd(z[vt], tt + vt * TT, re, im);
            else if constexpr (LOGM == 12) p1_fwd12(z[vt], tt + vt * TT, re, im);
            else p1_fwd11(z[vt], tt + vt * TT, re, im);
        }
    }
    // twiddle rows are requested ahead of each barrier; both virtual threads use the same row (TT is a multiple of 64)
    float2 gtw[8];
    if (fwd) tw_load8(&g_tw13.p2[0][tt & 63], 64, gtw);
    __syncthreads();
    if (fwd) {
#pragma unroll
        for (int vt = 0; vt < VT; ++vt) p2_fwd(tt + vt * TT, re, im, gtw);
    }
    // ---- per-unit constants of the pointwise stage ----
    const float* filt = a.filt + (size_t)d * a.filt_stride;
    const float2* hsrc = nullptr;
    int w_lo = 0x40000000, w_hi = -1;                      // empty band: no 32-bin window of pw_load overlaps it
    float cre = 0.f, cim = 0.f;
    double delta = 0.0;
    if (MODE == MODE_HDET) hsrc = a.h_det + (size_t)unit * K;
    if (MODE == MODE_FUSED) {
        const WfCoef* c = a.coef + b;
        hsrc = a.h0 + (size_t)b * K;
        if (c->valid) { w_lo = c->k_lo; w_hi = c->k_hi; }       // an empty band is stored as (2^30, -1) by prepare_kernel
        const DetResp r = a.resp[unit];
        cre = (float)r.fp * c->pol_p;                       // C = F+ (1+cos^2 i)/2 - i Fx cos i
        cim = -(float)r.fc * c->pol_c;
        delta = r.dt * (double)a.inv_tseg;                   // turns per bin (fp64: the second view's dt reaches 1 s)
    }
    // Operands of the pointwise stage for virtual thread t: bins k = t + KL k4 (half A) and M - k (half B), KL = 1024 (512).
    // They are requested one phase ahead of their use so that L2 latency is covered by butterfly work.  h0 is zero
    // outside [w_lo, w_hi]: a warp none of whose 32 bins of a half is inside skips the load (warp-uniform test;
    // heavy systems stop at a few hundred Hz).
    struct PwOps { float2 ha[8], hb[8]; float fa[8], fb[8]; };
    auto pw_load = [&](int t, PwOps& L) {
        const int wbase = t & ~31;
#pragma unroll
        for (int k4 = 0; k4 < 8; ++k4) {
            const int k = t + KL * k4;
            L.fa[k4] = __ldg(filt + k);
            L.fb[k4] = __ldg(filt + M - k);
            if (MODE == MODE_HDET) {
                L.ha[k4] = __ldg(hsrc + k);
                L.hb[k4] = __ldg(hsrc + M - k);
            } else if (MODE == MODE_FUSED) {
                const int ka_lo = wbase + KL * k4, ka_hi = ka_lo + 31;
                L.ha[k4] = make_float2(0.f, 0.f);
                L.hb[k4] = make_float2(0.f, 0.f);
                if (ka_hi >= w_lo && ka_lo <= w_hi) L.ha[k4] = __ldg(hsrc + k);
                if (M - ka_lo >= w_lo && M - ka_hi <= w_hi) L.hb[k4] = __ldg(hsrc + M - k);
            }
        }
    };
    auto inject = [&](int k, float2& x2) {                   // slow path (self-paired bins only)
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
    auto do_pair = [&](int k, float2& za, float2& zb) {       // za = Z[k], zb = Z[M-k], 0 < k <= M/2
        const float2 w = twiddle<N>(k);
        float2 xa, xb;
        split_pair(za, zb, w, xa, xb);
        inject(k, xa);
        inject(M - k, xb);
        const float fa = __ldg(filt + k), fb = __ldg(filt + M - k);
        xa.x *= fa; xa.y *= fa; xb.x *= fb; xb.y *= fb;
        merge_pair(xa, xb, w, za, zb);
    };
    __shared__ float2 sc[16];
    // a-7 inject, a-8 whiten + band-limit on the registers of virtual thread t (v[r]: k4 = brev(r); halves A, B)
    auto pointwise = [&](int t, C2 (&v)[8], const PwOps& L) {
        float2 za[8], zb[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            unpack(v[r].r, za[r].x, zb[r].x);
            unpack(v[r].i, za[r].y, zb[r].y);
        }
        // Thread 0 holds the two self-paired butterflies (klow 0: bins 1024 q, with DC/Nyquist in Z[0]; klow 512:
        // bins 512 + 1024 q).  It parks them in a scratch row; nine lanes of warp 0 process those bins after the
        // generic section (which thread 0 executes on values that are then overwritten), so no warp runs a long
        // divergent path.
        if (t == 0) {
#pragma unroll
            for (int r = 0; r < 8; ++r) { sc[brev<8>(r)] = za[r]; sc[8 + brev<8>(r)] = zb[r]; }
        }
        // split twiddle w_N^k = w_N^t * w_16^k4: one sincos and compile-time rotations.
        const float2 wt = twiddle<N>(t);
        // projection factors C exp(-2 pi i k dt/T) by recurrence over k4 (both halves in one packed chain):
        //   A: C e(t) e(1024)^k4,  B: C e(M) conj(e(t)) conj(e(1024))^k4,  e(j) = exp(-2 pi i j delta)
        C2 ph, st;
        if (MODE == MODE_FUSED) {
            auto unit_phase = [&](float turns) {
                turns -= rintf(turns);
                float s, co;
                __sincosf(turns * -6.283185307179586f, &s, &co);
                return make_float2(co, s);
            };
            float tt_, ts_, tm_;
            if (a.phase64) {                                 // second data view: dt reaches 1 s, reduce in fp64
                double x = (double)t * delta; tt_ = (float)(x - rint(x));
                x = (double)KL * delta; ts_ = (float)(x - rint(x));
                x = (double)M * delta; tm_ = (float)(x - rint(x));
            } else {                                         // |dt| <= 21 ms: fp32 is exact enough
                const float df = (float)delta;
                tt_ = (float)t * df; ts_ = (float)KL * df; tm_ = (float)M * df;
            }
            const float2 et = unit_phase(tt_);
            const float2 es = unit_phase(ts_);
            const float2 em = unit_phase(tm_);
            const float2 cc = make_float2(cre, cim);
            const float2 ca = amplfi::cmul(cc, et);
            const float2 cb = amplfi::cmul_conj(amplfi::cmul(cc, em), et);
            ph = C2{pack(ca.x, cb.x), pack(ca.y, cb.y)};
            st = C2{pack(es.x, es.x), pack(es.y, -es.y)};
        }
#pragma unroll
        for (int k4 = 0; k4 < 8; ++k4) {
            const int r = brev<8>(k4);
            float2 w = wt;
            switch (k4) {
                case 0: break;
                case 1: w = mul_w32<2, false>(wt); break;
                case 2: w = mul_w32<4, false>(wt); break;
                case 3: w = mul_w32<6, false>(wt); break;
                case 4: w = mul_w32<8, false>(wt); break;
                case 5: w = mul_w32<10, false>(wt); break;
                case 6: w = mul_w32<12, false>(wt); break;
                default: w = mul_w32<14, false>(wt); break;
            }
            float2& pa = za[r];
            float2& pb = zb[7 - r];
            float2 xa, xb;
            split_pair(pa, pb, w, xa, xb);
            const float2 ha = L.ha[k4], hb = L.hb[k4];
            if (MODE == MODE_HDET) {
                xa.x = fmaf(a.two_fs, ha.x, xa.x); xa.y = fmaf(a.two_fs, ha.y, xa.y);
                xb.x = fmaf(a.two_fs, hb.x, xb.x); xb.y = fmaf(a.two_fs, hb.y, xb.y);
            } else if (MODE == MODE_FUSED) {
                float ar, br, ai, bi;
                unpack(ph.r, ar, br);
                unpack(ph.i, ai, bi);
                xa.x = fmaf(ha.x, ar, fmaf(-ha.y, ai, xa.x));
                xa.y = fmaf(ha.x, ai, fmaf(ha.y, ar, xa.y));
                xb.x = fmaf(hb.x, br, fmaf(-hb.y, bi, xb.x));
                xb.y = fmaf(hb.x, bi, fmaf(hb.y, br, xb.y));
                if (k4 < 7) ph = cmul(ph, st);
            }
            const float fa = L.fa[k4], fb = L.fb[k4];
            xa.x *= fa; xa.y *= fa; xb.x *= fb; xb.y *= fb;
            merge_pair(xa, xb, w, pa, pb);
        }
        if (t < 32) {
            __syncwarp();
            if (t == 0) {       // Z[0] carries the DC and Nyquist bins of the real transform
                const float2 z0 = sc[0];
                float x0 = 2.0f * (z0.x + z0.y), xm = 2.0f * (z0.x - z0.y);
                if (MODE == MODE_HDET) {
                    x0 = fmaf(a.two_fs, __ldg(hsrc).x, x0);
                    xm = fmaf(a.two_fs, __ldg(hsrc + M).x, xm);
                }
                const float y0 = x0 * __ldg(filt), ym = xm * __ldg(filt + M);
                sc[0] = make_float2(y0 + ym, y0 - ym);
            } else if (t < 9) {
                // t = 1..3: (A[q], A[8-q]), k = 1024 q;  t = 4: A[4] with itself, k = M/2;
                // t = 5..8: (B[q], B[7-q]), q = t - 5, k = 512 + 1024 q
                const int ia = t <= 4 ? t : 3 + t, ib = t <= 4 ? 8 - t : 20 - t;
                const int k = t <= 4 ? KL * t : KL / 2 + KL * (t - 5);
                float2 pa = sc[ia], pb = sc[ib];
                do_pair(k, pa, pb);
                sc[ia] = pa;
                if (ib != ia) sc[ib] = pb;
            }
            __syncwarp();
            if (t == 0) {
#pragma unroll
                for (int r = 0; r < 8; ++r) { za[r] = sc[brev<8>(r)]; zb[r] = sc[8 + brev<8>(r)]; }
            }
        }
#pragma unroll
        for (int r = 0; r < 8; ++r) v[r] = C2{pack(za[r].x, zb[r].x), pack(za[r].y, zb[r].y)};
    };

    PwOps ops[VT];
    constexpr bool HOIST = (VIEWS == 1);                     // the two-view variant is short of registers: it requests after the barrier
    if (HOIST) {
        pw_load(tt, ops[0]);                                 // in flight during the barrier and P3
        if (fwd) tw_load8(&g_tw13.p3[0][tt & 7], 8, gtw);
    }
    __syncthreads();
    if (!HOIST) {
        pw_load(tt, ops[0]);
        if (fwd) tw_load8(&g_tw13.p3[0][tt & 7], 8, gtw);
    }
    if (fwd) {
#pragma unroll
        for (int vt = 0; vt < VT; ++vt) p3_fwd(tt + vt * TT, re, im, gtw);
    }
    __syncthreads();
    if constexpr (VIEWS == 2) {
        ulonglong2* stash = reinterpret_cast<ulonglong2*>(a.out2 + (size_t)unit * N);
        const double delta0 = delta;
        float2* outv = reinterpret_cast<float2*>(out);
#pragma unroll 1
        for (int view = 0; view < 2; ++view) {
            if (view == 1) {
                __syncthreads();                             // every thread is done reading smem for the first view
                delta = delta0 + a.t_shift[b] * (double)a.inv_tseg;
                outv = reinterpret_cast<float2*>(a.out2 + (size_t)unit * N);
                pw_load(tt, ops[0]);
            }
#pragma unroll
            for (int vt = 0; vt < VT; ++vt) {
                const int t = tt + vt * TT;
                const int klow_a = t, klow_b = (t == 0) ? KL / 2 : KL - t;
                C2 v[8];
                if (view == 0) {
                    p4_fwd<LOGM>(klow_a, klow_b, v, re, im);
#pragma unroll
                    for (int r = 0; r < 8; ++r) stash[r * G::T + t] = make_ulonglong2(v[r].r, v[r].i);
                } else {
#pragma unroll
                    for (int r = 0; r < 8; ++r) { const ulonglong2 q = stash[r * G::T + t]; v[r] = C2{q.x, q.y}; }
                }
                pointwise(t, v, ops[vt]);
                if (vt + 1 < VT) pw_load(t + TT, ops[vt + 1]);
                p4_inv<LOGM>(klow_a, klow_b, v, re, im);
            }
            __syncthreads();
            tw_load8(&g_tw13.p3i[0][tt & 63], 64, gtw);
#pragma unroll
            for (int vt = 0; vt < VT; ++vt) p3_inv(tt + vt * TT, re, im, gtw);
            __syncthreads();
#pragma unroll
            for (int vt = 0; vt < VT; ++vt) {                // (no hoisting here: this variant is short of registers)
                C2 tw2[8];
                p2_inv_twiddles<LOGM>(tt + vt * TT, tw2);
                p2_inv(tt + vt * TT, re, im, tw2);
            }
            __syncthreads();
#pragma unroll
            for (int vt = 0; vt < VT; ++vt) {
                float2 z[16];
                if constexpr (LOGM == 13) p1_inv(z, tt + vt * TT, re, im);
                else if constexpr (LOGM == 12) p1_inv12(z, tt + vt * TT, re, im);
                else p1_inv11(z, tt + vt * TT, re, im);
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1) __stcs(outv + sample_index<LOGM>(n1, tt + vt * TT), z[n1]);
            }
        }
        return;
    }
#pragma unroll
    for (int vt = 0; vt < VT; ++vt) {
        const int t = tt + vt * TT;
        const int klow_a = t, klow_b = (t == 0) ? KL / 2 : KL - t;
        C2 v[8];
        if (fwd) {
            p4_fwd<LOGM>(klow_a, klow_b, v, re, im);
        } else {
#pragma unroll
            for (int r = 0; r < 8; ++r) v[r] = C2{0ull, 0ull};
        }
        pointwise(t, v, ops[vt]);
        if (vt + 1 < VT) pw_load(t + TT, ops[vt + 1]);      // in flight during this P4' and the next P4
        // ---- a-9 inverse real FFT ----
        p4_inv<LOGM>(klow_a, klow_b, v, re, im);
    }
    tw_load8(&g_tw13.p3i[0][tt & 63], 64, gtw);
    __syncthreads();
#pragma unroll
    for (int vt = 0; vt < VT; ++vt) p3_inv(tt + vt * TT, re, im, gtw);
    C2 tw2[VT][8];
#pragma unroll
    for (int vt = 0; vt < VT; ++vt) p2_inv_twiddles<LOGM>(tt + vt * TT, tw2[vt]);
    __syncthreads();
#pragma unroll
    for (int vt = 0; vt < VT; ++vt) p2_inv(tt + vt * TT, re, im, tw2[vt]);
    __syncthreads();
    {
        float2* out2 = reinterpret_cast<float2*>(out);
#pragma unroll
        for (int vt = 0; vt < VT; ++vt) {
            float2 z[16];
            if constexpr (LOGM == 13) p1_inv(z, tt + vt * TT, re, im);
            else if constexpr (LOGM == 12) p1_inv12(z, tt + vt * TT, re, im);
            else p1_inv11(z, tt + vt * TT, re, im);
            if (a.crop == 0) {
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1) __stcs(out2 + sample_index<LOGM>(n1, tt + vt * TT), z[n1]);
            } else {
                const int c2 = a.crop >> 1;                  // crop is even: whole float2 pairs
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1) {
                    const int m = sample_index<LOGM>(n1, tt + vt * TT);
                    if (m >= c2 && m < M - c2) __stcs(out2 + m - c2, z[n1]);
                }
            }
        }
    }
}


__global__ void init_tw13_kernel() {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;       // 0 .. 511
    auto w = [](int num, int den) {                           // exp(-2 pi i num / den), fp64 -> fp32
        double s, c;
        sincospi(-2.0 * (double)(num % den) / (double)den, &s, &c);
        return make_float2((float)c, (float)s);
    };
    auto put = [](float4& dst, int k, float2 v) { if (k & 1) { dst.z = v.x; dst.w = v.y; } else { dst.x = v.x; dst.y = v.y; } };
    if (i < 512) {
        const int s = i >> 3, k = i & 7;                       // p2: set s, power k
        put(g_tw13.p2[k >> 1][s], k, w(s * k, 512));
        const int k2 = s >> 3, n4 = s & 7, n3 = k;             // p3i: set s = k2*8 + n4, entry n3
        put(g_tw13.p3i[n3 >> 1][s], n3, w((n3 * 8 + n4) * k2, 512));
    }
    if (i < 64) {
        const int n4 = i >> 3, k = i & 7;
        put(g_tw13.p3[k >> 1][n4], k, w(n4 * k, 64));
        const int c = i >> 3, m4 = i & 7;                      // p4i: combination c, time digit m4
        const int k3a = c >> 1;
        for (int lg = 0; lg < 3; ++lg) {                       // LOGM = 11 + lg: klow >> s3 = k3, klow spans kl
            const int s3 = 5 + lg, kl = 256 << lg;
            const int t = (k3a << s3) + (c & 1);               // a representative thread of the combination
            const int klow_b = (t == 0) ? kl / 2 : kl - t;
            const float2 A = w(m4 * k3a, 64), B = w(m4 * (klow_b >> s3), 64);
            g_tw13.p4i[lg][c][m4] = make_ulonglong2(pack(A.x, B.x), pack(A.y, B.y));
        }
    }
}

// Once per device: the tables are the same for every plan, and amplfi_plan_create synchronises before it returns, so a
// later plan never rewrites them under a running kernel of an earlier one.
int init_iw13_tables(cudaStream_t st) {
    static std::atomic<unsigned> done{0};
    int dev = 0;
    cudaGetDevice(&dev);
    const unsigned bit = 1u << (dev & 31);
    if (done.load(std::memory_order_acquire) & bit) return AMPLFI_OK;
    init_tw13_kernel<<<2, 256, 0, st>>>();
    count_launch();
    const int rc = check_launch("init_tw13_kernel");
    if (rc) return rc;
    if (cudaStreamSynchronize(st) != cudaSuccess) { set_error("init_tw13_kernel: synchronise failed"); return AMPLFI_ERR_CUDA; }
    done.fetch_or(bit, std::memory_order_release);
    return AMPLFI_OK;
}

#ifndef IW13_VT
#define IW13_VT 2
#endif
template <int LOGM, int MODE, bool FWD, int VIEWS = 1>
static int launch_iw13_t(const IwArgs& a, int units, cudaStream_t st) {
    static std::atomic<unsigned> attr_done{0};
    constexpr int T13 = Geo<LOGM>::T;
    const int smem = 2 * Geo<LOGM>::M * (int)sizeof(float);
    const int rc = ensure_dynamic_smem(inject_whiten13_kernel<LOGM, MODE, IW13_VT, FWD, VIEWS>, smem, attr_done);
    if (rc) return rc;
    inject_whiten13_kernel<LOGM, MODE, IW13_VT, FWD, VIEWS><<<units, T13 / IW13_VT, smem, st>>>(a, units);
    count_launch();
    return check_launch("inject_whiten13_kernel");
}

template <int LOGM>
static int launch_iw13_l(const IwArgs& a, int mode, int units, cudaStream_t st) {
    // only the one-launch two-view call still runs this kernel (every single-view launch of n = 4096, 8192, 16384 goes to
    // inject_whiten_v3.cu)
    if (a.out2 == nullptr || mode != MODE_FUSED || a.noise == nullptr || a.t_shift == nullptr || a.crop != 0) {
        set_error("inject_whiten13: the two-view launch needs the fused mode");
        return AMPLFI_ERR_INVALID_ARG;
    }
    return launch_iw13_t<LOGM, MODE_FUSED, true, 2>(a, units, st);
}

int launch_iw13(const IwArgs& a, int logm, int mode, int units, cudaStream_t st) {
    if (logm == 13) return launch_iw13_l<13>(a, mode, units, st);
    if (logm == 12) return launch_iw13_l<12>(a, mode, units, st);
    return launch_iw13_l<11>(a, mode, units, st);
}

}  // namespace amplfi
