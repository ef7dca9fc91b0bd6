// waveform.cu -- per-sample preparation, materialised waveform and projection kernels.
// PAPER.md:87, :104 (waveform on the GPU), PAPER.md:190 (antenna response on the fly).
#include "amplfi_internal.h"
#include "spec_layout.cuh"
#include "waveform.cuh"

namespace amplfi {

// ---- plan tables: k^(-1/3) and ln k in fp64 ----
__global__ void tables_kernel(double* __restrict__ ci, double* __restrict__ lnk, int n_bins) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_bins) return;
    if (k == 0) { ci[0] = 0.0; lnk[0] = 0.0; return; }
    const double kd = (double)k;
    ci[k] = 1.0 / cbrt(kd);
    lnk[k] = log(kd);
}

int launch_tables(amplfi_plan* p, cudaStream_t st) {
    tables_kernel<<<(p->n_bins + 255) / 256, 256, 0, st>>>(p->tab_ci, p->tab_lnk, p->n_bins);
    count_launch();
    return check_launch("tables_kernel");
}

// ---- per sample: waveform coefficients and detector responses, fp64 ----
// All three are long dependent chains of fp64 arithmetic and library calls; a CTA of 96 threads serves 32 samples, warp 0
// computing the phase coefficients, warp 1 the amplitude coefficients (waveform.cuh: the two roles of prepare_sample, each
// writing its own fields of WfCoef) and warp 2 the responses, so the three chains run side by side on different schedulers.
__device__ __forceinline__ void store_phase_fields(WfCoef* __restrict__ o, const WfCoef& c) {
    o->valid = c.valid; o->approx = c.approx; o->k_lo = c.k_lo; o->k_hi = c.k_hi;
    o->kp1 = c.kp1; o->kp2 = c.kp2;
    o->lin1 = c.lin1; o->c01 = c.c01; o->a_m5 = c.a_m5; o->a_m3 = c.a_m3; o->a_m2 = c.a_m2; o->a_m1 = c.a_m1; o->a_ln = c.a_ln;
    o->a_p1 = c.a_p1; o->a_p1ln = c.a_p1ln; o->a_p2 = c.a_p2; o->s_p4 = c.s_p4; o->s_p5 = c.s_p5; o->s_p6 = c.s_p6;
    o->lin2 = c.lin2; o->c02 = c.c02; o->b_ln = c.b_ln; o->b_m9 = c.b_m9;
    o->lin3 = c.lin3; o->c03 = c.c03; o->r_m3 = c.r_m3; o->r_34 = c.r_34;
    o->r_at = c.r_at; o->at_k0 = c.at_k0; o->at_invw = c.at_invw;
    o->pol_p = c.pol_p; o->pol_c = c.pol_c;
}
__device__ __forceinline__ void store_amp_fields(WfCoef* __restrict__ o, const WfCoef& c) {
    o->amp_scale = c.amp_scale; o->ka1 = c.ka1; o->ka2 = c.ka2;
#pragma unroll
    for (int i = 0; i < 8; ++i) o->e[i] = c.e[i];
#pragma unroll
    for (int i = 0; i < 5; ++i) o->q[i] = c.q[i];
    o->q_mid = c.q_mid; o->q_invh = c.q_invh;
    o->g0 = c.g0; o->g_krd = c.g_krd; o->g_invw = c.g_invw; o->g2 = c.g2;
}

__global__ void __launch_bounds__(96) prepare_kernel(const double* __restrict__ params, int batch, int approx, double t_seg,
                                                     int n_bins, double f_lo, double f_hi, double amp_mul, double gmst,
                                                     const double* __restrict__ pd_table, const int* __restrict__ det_ids,
                                                     int n_det, WfCoef* __restrict__ coef, DetResp* __restrict__ resp,
                                                     int* __restrict__ flags) {
    const int b = blockIdx.x * 32 + (threadIdx.x & 31);
    if (b >= batch) return;
    const double* p = params + (size_t)b * AMPLFI_N_PARAMS;
    const int role = threadIdx.x >> 5;
    if (role == 0) {
        if (coef != nullptr) {
            WfCoef c;
            prepare_sample<WF_PHASE>(p, approx, t_seg, n_bins, f_lo, f_hi, amp_mul, pd_table, c);
            // canonical empty band: no 32-bin window of the fused kernel's operand loads may overlap it
            if (c.k_lo > c.k_hi) { c.k_lo = 0x40000000; c.k_hi = -1; }
            store_phase_fields(coef + b, c);
            if (flags != nullptr) flags[b] = c.valid ? 0 : 1;
        }
    } else if (role == 1) {
        if (coef != nullptr) {
            WfCoef c;
            prepare_sample<WF_AMP>(p, approx, t_seg, n_bins, f_lo, f_hi, amp_mul, pd_table, c);
            store_amp_fields(coef + b, c);
        }
    } else {
        const SkyFrame f = sky_frame(p[8], p[9], p[10], gmst);
        for (int d = 0; d < n_det; ++d) resp[(size_t)b * n_det + d] = detector_response(f, det_ids[d]);
    }
}

int launch_prepare(const amplfi_plan* p, int approximant, int batch, const double* params, double gmst,
                   double f_lo, double f_hi, double amp_mul, int* flags, cudaStream_t st) {
    if (approximant >= 0) p->last_approx = approximant;     // selects the evaluation kernel that follows
    prepare_kernel<<<(batch + 31) / 32, 96, 0, st>>>(
        params, batch, approximant, p->t_seg, p->n_bins, f_lo, f_hi, amp_mul, gmst, p->pd_table, p->d_det_ids,
        p->n_det, approximant < 0 ? nullptr : p->coef, p->resp, flags);
    count_launch();
    return check_launch("prepare_kernel");
}

// ---- materialised polarisations: hp = (1+cos^2 i)/2 h0, hc = -i cos i h0 ----
// gridDim.x CTAs share one sample and take its 256-bin chunks round-robin; the coefficient struct is staged once
// per CTA and chunks entirely outside the band [k_lo, k_hi] (common: heavy systems stop at a few hundred Hz) are
// zero-filled without touching the tables.
#define WF_SLICES 2
template <bool POL>
__global__ void __launch_bounds__(256, 4) waveform_kernel(const WfCoef* __restrict__ coef, const double* __restrict__ tab_ci,
                                                       const double* __restrict__ tab_lnk, int n_bins,
                                                       float2* __restrict__ out_a, float2* __restrict__ out_b) {
    const int b = blockIdx.y;
    __shared__ WfCoef c;
    {
        const int* src = reinterpret_cast<const int*>(coef + b);
        int* dst = reinterpret_cast<int*>(&c);
        if (threadIdx.x < (int)(sizeof(WfCoef) / sizeof(int))) dst[threadIdx.x] = src[threadIdx.x];
    }
    __syncthreads();
    const int k_lo = c.valid ? c.k_lo : 1, k_hi = c.valid ? c.k_hi : 0;
    float2* oa = out_a + (size_t)b * n_bins;
    float2* ob = POL ? out_b + (size_t)b * n_bins : nullptr;
    // The plan's h0 workspace (POL == false) is only ever read inside the band, widened to the 32-bin windows of
    // the consumers' warp-uniform band test: bins further than 64 from the band are not written.
    int k_first = 0, k_last = n_bins - 1;
    if (!POL) {
        if (k_lo > k_hi) return;
        k_first = k_lo > 64 ? ((k_lo - 64) & ~255) : 0;
        k_last = k_hi + 64 < n_bins - 1 ? k_hi + 64 : n_bins - 1;
    }
    // the table values of the next chunk are requested before the current chunk is evaluated (L2 latency off the chain)
    const int kstep = 256 * gridDim.x;
    int k = k_first + blockIdx.x * 256 + threadIdx.x;
    bool in = k >= k_lo && k <= k_hi;
    double ci = in ? tab_ci[k] : 1.0, lnk = in ? tab_lnk[k] : 0.0;
    for (; k <= k_last; k += kstep) {
        const int kn = k + kstep;
        const bool in_n = kn >= k_lo && kn <= k_hi;
        const double ci_n = in_n ? tab_ci[kn] : 1.0, lnk_n = in_n ? tab_lnk[kn] : 0.0;
        float2 h = make_float2(0.f, 0.f);
        if (in) h = eval_h0(c, k, ci, lnk);
        if (POL) {
            oa[k] = make_float2(c.pol_p * h.x, c.pol_p * h.y);
            ob[k] = make_float2(c.pol_c * h.y, -c.pol_c * h.x);     // -i c (x + i y) = c y - i c x
        } else {
            oa[k] = h;
        }
        in = in_n; ci = ci_n; lnk = lnk_n;
    }
}

// ---- sine-Gaussian family: a closed form per bin, no tables (its own small kernel so that the tuned kernel above is
// not touched); same outputs and the same "written only near the band" rule for the h0 workspace ----
template <bool POL>
__global__ void __launch_bounds__(256) sine_gaussian_kernel(const WfCoef* __restrict__ coef, int n_bins,
                                                            float2* __restrict__ out_a, float2* __restrict__ out_b) {
    const int b = blockIdx.y;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_bins) return;
    const WfCoef& c = coef[b];
    const bool in = c.valid && k >= c.k_lo && k <= c.k_hi;
    if (!POL && !in && (!c.valid || k < c.k_lo - 64 || k > c.k_hi + 64)) return;
    const float2 h = in ? eval_sine_gaussian(c, k) : make_float2(0.f, 0.f);
    if (POL) {
        out_a[(size_t)b * n_bins + k] = make_float2(c.pol_p * h.x, c.pol_p * h.y);
        out_b[(size_t)b * n_bins + k] = make_float2(c.pol_c * h.y, -c.pol_c * h.x);
    } else {
        out_a[(size_t)b * n_bins + k] = h;
    }
}


// ---- h0 in the slot layout of the n = 16384 fused kernel (spec_layout.cuh) ----
// gridDim.x CTAs share one sample and take its 16 slot groups (second, w) round-robin; a warp skips the groups that
// slot::window_needed() does not mark (the consumer skips exactly those).  Thread t produces whole 16-byte slots: the
// two bins of a slot are evaluated one after the other by ONE copy of the evaluation code (64 registers, four CTAs per
// SM: the kernel is bound by the latency of the fp64 phase chain, so resident warps count), the table values of the next
// bin requested before the current one is evaluated; bins outside the band are written as exact zeros.
template <int FAMILY>       // 0: TaylorF2 / IMRPhenomD (power tables), 1: sine-Gaussian (closed form)
__global__ void __launch_bounds__(512, 2) waveform_slots_kernel(const WfCoef* __restrict__ coef, const double* __restrict__ tab_ci,
                                                                const double* __restrict__ tab_lnk, float* __restrict__ h0, int kl) {
    // kl / 2 threads per sample (the consumer's thread count), in gridDim.z blocks of at most 512
    const int b = blockIdx.y, t = blockIdx.z * blockDim.x + threadIdx.x, wi = t >> 5, nt = kl >> 1;
    __shared__ WfCoef c;
    {
        const int* src = reinterpret_cast<const int*>(coef + b);
        int* dst = reinterpret_cast<int*>(&c);
        constexpr int NW = (int)(sizeof(WfCoef) / sizeof(int));           // 78 words; CTAs have 64 .. 512 threads
        static_assert(NW <= 128, "two rounds of a 64-thread CTA must cover WfCoef");
        const int q = threadIdx.x;
        if (q < NW) dst[q] = src[q];
        if (q + 64 < NW && blockDim.x == 64) dst[q + 64] = src[q + 64];
    }
    __syncthreads();
    if (!c.valid || c.k_lo > c.k_hi) return;
    const int k_lo = c.k_lo, k_hi = c.k_hi;
    float4* row = reinterpret_cast<float4*>(h0 + (size_t)b * slot::h0_row(kl)) + t;
    // groups of this warp: bit g = second * 8 + w set iff the consumer reads it (one ballot instead of a test per group);
    // the CTAs of a sample share them round-robin
    const int lane_id = t & 31;
    // (gridDim.x is 2, 4 or 8: launch_waveform_h0)
    unsigned todo = __ballot_sync(0xffffffffu, lane_id < 16 && (lane_id & (gridDim.x - 1)) == blockIdx.x &&
                                                   slot::window_needed(kl, lane_id >> 3, lane_id & 7, wi, k_lo, k_hi));
#pragma unroll 1
    while (todo) {
        const int g = __ffs(todo) - 1;
        todo &= todo - 1;
        int kA, kB;
        slot::slot_bins(kl, g >> 3, g & 7, t, kA, kB);
        const bool inA = kA >= k_lo && kA <= k_hi, inB = kB >= k_lo && kB <= k_hi;
        // the table values of both bins are requested together (one L2 round trip per slot)
        double ciA = 1.0, lnA = 0.0, ciB = 1.0, lnB = 0.0;
        if (FAMILY == 0) {
            if (inA) { ciA = tab_ci[kA]; lnA = tab_lnk[kA]; }
            if (inB) { ciB = tab_ci[kB]; lnB = tab_lnk[kB]; }
        }
        float2 hA = make_float2(0.f, 0.f), hB = make_float2(0.f, 0.f);
#pragma unroll
        for (int lane = 0; lane < 2; ++lane) {
            const int k = lane ? kB : kA;
            float2 h = make_float2(0.f, 0.f);
            if (lane ? inB : inA) {
                if (FAMILY == 0) h = eval_h0(c, k, lane ? ciB : ciA, lane ? lnB : lnA);
                else h = eval_sine_gaussian(c, k);
            }
            if (lane) hB = h; else hA = h;
        }
        row[g * nt] = make_float4(hA.x, hB.x, hA.y, hB.y);
    }
}

int launch_waveform_pol(const amplfi_plan* p, int batch, float* hp, float* hc, cudaStream_t st) {
    if (p->last_approx == 2) {
        dim3 g((p->n_bins + 255) / 256, batch);
        sine_gaussian_kernel<true><<<g, 256, 0, st>>>(p->coef, p->n_bins, reinterpret_cast<float2*>(hp),
                                                      reinterpret_cast<float2*>(hc));
        count_launch();
        return check_launch("sine_gaussian_kernel<pol>");
    }
    dim3 grid(WF_SLICES, batch);
    waveform_kernel<true><<<grid, 256, 0, st>>>(p->coef, p->tab_ci, p->tab_lnk, p->n_bins,
                                                reinterpret_cast<float2*>(hp), reinterpret_cast<float2*>(hc));
    count_launch();
    return check_launch("waveform_kernel<pol>");
}

int launch_waveform_h0(const amplfi_plan* p, int batch, cudaStream_t st, int slots) {
    if (slots) {            // slot layout of the three-pass fused kernel (n = 4096 .. 131072)
        const int kl = p->n / 32;
        const int nthr = kl / 2 > 512 ? 512 : kl / 2;
        dim3 grid(batch >= 1024 ? 2 : (batch >= 64 ? 4 : 8), batch, (kl / 2) / nthr);
        float* h0f = reinterpret_cast<float*>(p->h0);
        if (p->last_approx == 2) waveform_slots_kernel<1><<<grid, nthr, 0, st>>>(p->coef, p->tab_ci, p->tab_lnk, h0f, kl);
        else waveform_slots_kernel<0><<<grid, nthr, 0, st>>>(p->coef, p->tab_ci, p->tab_lnk, h0f, kl);
        count_launch();
        return check_launch("waveform_slots_kernel");
    }
    if (p->last_approx == 2) {
        dim3 g((p->n_bins + 255) / 256, batch);
        sine_gaussian_kernel<false><<<g, 256, 0, st>>>(p->coef, p->n_bins, p->h0, nullptr);
        count_launch();
        return check_launch("sine_gaussian_kernel<h0>");
    }
    // (long segments come in small batches: more CTAs per sample then, up to about eight resident CTAs per SM)
    int slices = (8 * p->sm_count) / (batch > 0 ? batch : 1);
    slices = slices < WF_SLICES ? WF_SLICES : (slices > 64 ? 64 : slices);
    dim3 grid(slices, batch);
    waveform_kernel<false><<<grid, 256, 0, st>>>(p->coef, p->tab_ci, p->tab_lnk, p->n_bins, p->h0, nullptr);
    count_launch();
    return check_launch("waveform_kernel<h0>");
}

// ---- projection: h_d = (F+ h+ + Fx hx) exp(-2 pi i f_k dt_d) ----
__global__ void __launch_bounds__(256) project_kernel(const DetResp* __restrict__ resp, int n_det, int n_bins,
                                                      double inv_tseg, const float2* __restrict__ hp,
                                                      const float2* __restrict__ hc, float2* __restrict__ h_det) {
    const int b = blockIdx.y;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_bins) return;
    const float2 p = hp[(size_t)b * n_bins + k];
    const float2 c = hc[(size_t)b * n_bins + k];
    for (int d = 0; d < n_det; ++d) {
        const DetResp r = resp[(size_t)b * n_det + d];
        const float fp = (float)r.fp, fc = (float)r.fc;
        const float2 h = make_float2(fp * p.x + fc * c.x, fp * p.y + fc * c.y);
        double turns = (double)k * (r.dt * inv_tseg);
        turns -= rint(turns);
        float s, co;
        sincospif(2.0f * (float)turns, &s, &co);
        // h * (cos - i sin)
        h_det[((size_t)b * n_det + d) * n_bins + k] = make_float2(h.x * co + h.y * s, h.y * co - h.x * s);
    }
}

// ---- second data view: same responses, arrival time later by t_shift[b] ----
__global__ void shift_resp_kernel(const DetResp* __restrict__ resp, const double* __restrict__ t_shift, int n_det, int count,
                                  DetResp* __restrict__ resp2) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    DetResp r = resp[i];
    r.dt += t_shift[i / n_det];
    resp2[i] = r;
}

int launch_shift_resp(const amplfi_plan* p, int batch, const double* t_shift, cudaStream_t st) {
    const int count = batch * p->n_det;
    shift_resp_kernel<<<(count + 127) / 128, 128, 0, st>>>(p->resp, t_shift, p->n_det, count, p->resp2);
    count_launch();
    return check_launch("shift_resp_kernel");
}

// ---- the two polarisations as pseudo-detectors: (F+, Fx, dt) = (1, 0, 0) and (0, 1, 0) (amplfi_waveform_td) ----
__global__ void td_resp_kernel(int count, DetResp* __restrict__ resp2) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    DetResp r;
    r.fp = (i & 1) ? 0.0 : 1.0;
    r.fc = (i & 1) ? 1.0 : 0.0;
    r.dt = 0.0;
    resp2[i] = r;
}

int launch_td_resp(const amplfi_plan* p, int batch, cudaStream_t st) {
    const int count = batch * 2;
    td_resp_kernel<<<(count + 127) / 128, 128, 0, st>>>(count, p->resp2);
    count_launch();
    return check_launch("td_resp_kernel");
}

__global__ void copy_resp_kernel(const DetResp* __restrict__ resp, double* __restrict__ out, int count) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    out[3 * i + 0] = resp[i].fp;
    out[3 * i + 1] = resp[i].fc;
    out[3 * i + 2] = resp[i].dt;
}

int launch_project(const amplfi_plan* p, int batch, const float* hp, const float* hc, float* h_det,
                   double* resp_out, cudaStream_t st) {
    if (h_det != nullptr) {
        dim3 grid((p->n_bins + 255) / 256, batch);
        project_kernel<<<grid, 256, 0, st>>>(p->resp, p->n_det, p->n_bins, 1.0 / p->t_seg,
                                             reinterpret_cast<const float2*>(hp), reinterpret_cast<const float2*>(hc),
                                             reinterpret_cast<float2*>(h_det));
        count_launch();
        int rc = check_launch("project_kernel");
        if (rc) return rc;
    }
    if (resp_out != nullptr) {
        const int count = batch * p->n_det;
        copy_resp_kernel<<<(count + 127) / 128, 128, 0, st>>>(p->resp, resp_out, count);
        count_launch();
        return check_launch("copy_resp_kernel");
    }
    return AMPLFI_OK;
}

}  // namespace amplfi
