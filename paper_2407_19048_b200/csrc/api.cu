// api.cu -- the C ABI of libamplfi (include/amplfi.h): argument validation, plan management and the
// sequencing of kernel launches.  No computation happens on the host.
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "amplfi_internal.h"
#include "fft_core.cuh"
#include "waveform.cuh"

namespace amplfi {

static thread_local char g_err[512] = "";
static std::atomic<long> g_launches{0};

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int check_launch(const char* what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        set_error("%s: %s", what, cudaGetErrorString(e));
        return AMPLFI_ERR_CUDA;
    }
    return AMPLFI_OK;
}

static bool is_pow2_in_range(long v, long hi = 65536) { return v >= 1024 && v <= hi && (v & (v - 1)) == 0; }

static const double kPdTable[AMPLFI_PD_ROWS][AMPLFI_PD_COLS] = AMPLFI_PD_TABLE_INIT;

template <class T>
static int dev_alloc(T** ptr, size_t count) {
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(ptr), count * sizeof(T));
    if (e != cudaSuccess) {
        set_error("cudaMalloc(%zu bytes): %s", count * sizeof(T), cudaGetErrorString(e));
        return AMPLFI_ERR_CUDA;
    }
    return AMPLFI_OK;
}

// segment lengths of the three-pass fused kernel (inject_whiten_v3.cu), whose h0 workspace is in the slot layout
static bool v3_family(const amplfi_plan* p) { return p->logm >= 11 && p->logm <= 16; }

static bool known_approximant(int a) { return a == AMPLFI_TAYLORF2 || a == AMPLFI_IMRPHENOMD || a == AMPLFI_SINE_GAUSSIAN; }

// a plan's tables and workspaces live on the device it was created on
static int check_device(const amplfi_plan* p, const char* who) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) {
        set_error("%s: the plan belongs to device %d, the current device is %d", who, p->device, dev);
        return AMPLFI_ERR_INVALID_ARG;
    }
    return AMPLFI_OK;
}

static int validate_band(const amplfi_plan* p, double f_lo, double f_hi, const char* who) {
    const int rcd = check_device(p, who);
    if (rcd) return rcd;
    if (!(f_lo >= 0.0) || !(f_hi > f_lo) || !(f_hi <= 0.5 * p->fs)) {
        set_error("%s: need 0 <= f_lo < f_hi <= fs/2 (got %g, %g, fs %g)", who, f_lo, f_hi, p->fs);
        return AMPLFI_ERR_INVALID_ARG;
    }
    return AMPLFI_OK;
}

}  // namespace amplfi

using namespace amplfi;

// ---- fp32 pipe probe (amplfi_probe_fp32_pipe) ----
__global__ void __launch_bounds__(256) fp32_probe_kernel(unsigned long long* out, unsigned long long a, unsigned long long b,
                                                         int iters) {
    unsigned long long x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = (unsigned long long)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[i]) : "l"(a), "l"(b));
    }
    unsigned long long s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void fill_kernel(float* dst, int count, float v) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) dst[i] = v;
}

extern "C" int amplfi_probe_fp32_pipe(double* lane_ops_per_s) {
    if (lane_ops_per_s == nullptr) { set_error("amplfi_probe_fp32_pipe: null pointer"); return AMPLFI_ERR_INVALID_ARG; }
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    unsigned long long* buf = nullptr;
    const int ctas = sms * 8, iters = 4096;
    if (e == cudaSuccess) e = cudaMalloc(&buf, (size_t)ctas * 256 * sizeof(unsigned long long));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    float best = 0.f;
    if (e == cudaSuccess) {
        const unsigned long long a = 0x3f8000013f800001ull, b = 0x3089705f3089705full;     // (1 + 2^-23, ~1e-9) x 2
        for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {                             // first pass warms up
            cudaEventRecord(e0, nullptr);
            fp32_probe_kernel<<<ctas, 256>>>(buf, a, b, iters);
            cudaEventRecord(e1, nullptr);
            e = cudaEventSynchronize(e1);
            float ms = 0.f;
            if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms > 0.f && (best == 0.f || ms < best)) best = ms;
        }
        count_launch(4);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess || best <= 0.f) { set_error("amplfi_probe_fp32_pipe: %s", cudaGetErrorString(e)); return AMPLFI_ERR_CUDA; }
    *lane_ops_per_s = (double)ctas * 256.0 * 8.0 * iters * 2.0 / ((double)best * 1e-3);
    return AMPLFI_OK;
}

extern "C" {

const char* amplfi_last_error(void) { return g_err; }

double amplfi_psd_scale(void) { return std::ldexp(1.0, 140); }

const char* amplfi_version(void) { return "amplfi-b200 0.1 (sm_100a)"; }

long amplfi_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int amplfi_phenomd_table(double* out) {
    if (out == nullptr) { set_error("amplfi_phenomd_table: null output"); return AMPLFI_ERR_INVALID_ARG; }
    std::memcpy(out, kPdTable, sizeof(kPdTable));
    return AMPLFI_OK;
}

int amplfi_qnm_table(double* out) {
    if (out == nullptr) { set_error("amplfi_qnm_table: null output"); return AMPLFI_ERR_INVALID_ARG; }
    const double* qnm = kerr_qnm_table();
    if (qnm == nullptr) { set_error("amplfi_qnm_table: the continued-fraction iteration did not converge"); return AMPLFI_ERR_CUDA; }
    std::memcpy(out, qnm, sizeof(double) * 2 * AMPLFI_QNM_NODES);
    return AMPLFI_QNM_NODES;
}

int amplfi_plan_create(int n, double fs, int n_det, const int* det_ids, int max_batch, int nperseg,
                       amplfi_plan** out) {
    if (out == nullptr || det_ids == nullptr) { set_error("amplfi_plan_create: null pointer"); return AMPLFI_ERR_INVALID_ARG; }
    *out = nullptr;
    if (n_det < 1 || n_det > 3 || max_batch < 1 || !(fs > 0.0) || !std::isfinite(fs)) {
        set_error("amplfi_plan_create: need 1 <= n_det <= 3, max_batch >= 1, fs > 0");
        return AMPLFI_ERR_INVALID_ARG;
    }
    for (int d = 0; d < n_det; ++d)
        if (det_ids[d] < 0 || det_ids[d] > 2) { set_error("amplfi_plan_create: unknown detector id %d", det_ids[d]); return AMPLFI_ERR_INVALID_ARG; }
    if (!is_pow2_in_range(n, 1L << 20)) { set_error("amplfi_plan_create: n = %d is not a power of two in [2^10, 2^20]", n); return AMPLFI_ERR_UNSUPPORTED_SIZE; }
    if (nperseg != 0 && (!is_pow2_in_range(nperseg) || nperseg > 32768)) {
        set_error("amplfi_plan_create: nperseg = %d is not a power of two in [2^10, 2^15]", nperseg);
        return AMPLFI_ERR_UNSUPPORTED_SIZE;
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    int sms = 0;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { set_error("amplfi_plan_create: no CUDA device (%s)", cudaGetErrorString(e)); return AMPLFI_ERR_CUDA; }

    amplfi_plan* p = new amplfi_plan();
    std::memset(p, 0, sizeof(*p));
    p->n = n; p->n_bins = n / 2 + 1; p->logm = ilog2(n) - 1;
    p->fs = fs; p->t_seg = (double)n / fs;
    p->n_det = n_det;
    for (int d = 0; d < n_det; ++d) p->det_ids[d] = det_ids[d];
    p->max_batch = max_batch; p->nperseg = nperseg; p->device = dev; p->sm_count = sms;
    p->welch_max_seg = 256;
    int rc = AMPLFI_OK;
    if (!rc) rc = dev_alloc(&p->tab_ci, (size_t)p->n_bins);
    if (!rc) rc = dev_alloc(&p->tab_lnk, (size_t)p->n_bins);
    if (!rc) rc = dev_alloc(&p->pd_table, (size_t)AMPLFI_QNM_OFFSET + 2 * AMPLFI_QNM_NODES);
    if (!rc) rc = dev_alloc(&p->coef, (size_t)max_batch);
    if (!rc) rc = dev_alloc(&p->resp, (size_t)max_batch * n_det);
    if (!rc) rc = dev_alloc(&p->resp2, (size_t)max_batch * 3);
    if (!rc) rc = dev_alloc(&p->h0, (size_t)max_batch * p->n_bins);
    p->filt_stride = (p->n_bins + 3) & ~3;
    if (!rc) rc = dev_alloc(&p->filt, (size_t)n_det * p->filt_stride);
    if (!rc && p->logm >= 11 && p->logm <= 16) rc = dev_alloc(&p->filt_slots, (size_t)n_det * (n / 2));
    if (!rc) rc = dev_alloc(&p->filt_flat, (size_t)p->filt_stride);
    if (!rc) rc = dev_alloc(&p->fir_spec, (size_t)n_det * p->n_bins);
    if (!rc) rc = dev_alloc(&p->fir_time, (size_t)n_det * n);
    if (!rc) rc = dev_alloc(&p->d_det_ids, (size_t)3);
    if (!rc && p->logm >= 17) {
        // four-step path (inject_whiten_long.cu): n/32768 + 1 rows of 16384 complex points per unit, one CTA per row and SM;
        // a chunk is two full waves of rows and its scratch (39 MB) stays in L2
        const int rdec = n / 16384, rows = rdec / 2 + 1;
        // units per chunk: the count (scratch <= 64 MB) whose rows fill whole waves of SMs best
        const int nsm = sms > 0 ? sms : 148;
        const int umax = (int)((64u << 20) / ((size_t)rows * 16384 * 8));
        double best = 0.0;
        p->long_chunk = 1;
        for (int u = 1; u <= (umax < 1 ? 1 : umax); ++u) {
            const int ctas = u * rows, waves = (ctas + nsm - 1) / nsm;
            const double util = (double)ctas / ((double)waves * nsm);
            if (util >= best) { best = util; p->long_chunk = u; }
        }
        rc = dev_alloc(&p->long_spec, amplfi::long_scratch_floats2(p->long_chunk, rdec));
        if (!rc) rc = dev_alloc(&p->long_filt_rows, (size_t)3 * amplfi::long_row_elems(rdec));
        if (!rc) rc = dev_alloc(&p->long_h0_rows, (size_t)max_batch * amplfi::long_row_elems(rdec));
    }
    if (!rc && nperseg) rc = dev_alloc(&p->welch_part, (size_t)n_det * p->welch_max_seg * (nperseg / 2 + 1));
    if (!rc) {
        e = cudaMemcpy(p->pd_table, kPdTable, sizeof(kPdTable), cudaMemcpyHostToDevice);
        const double* qnm = kerr_qnm_table();
        if (qnm == nullptr) { set_error("amplfi_plan_create: the Kerr quasi-normal-mode table did not converge"); rc = AMPLFI_ERR_CUDA; }
        else if (e == cudaSuccess) e = cudaMemcpy(p->pd_table + AMPLFI_QNM_OFFSET, qnm, sizeof(double) * 2 * AMPLFI_QNM_NODES, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(p->d_det_ids, p->det_ids, sizeof(int) * 3, cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { set_error("amplfi_plan_create: cudaMemcpy: %s", cudaGetErrorString(e)); rc = AMPLFI_ERR_CUDA; }
    }
    if (!rc) {
        e = cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming);
        if (e != cudaSuccess) { set_error("amplfi_plan_create: stream/event: %s", cudaGetErrorString(e)); rc = AMPLFI_ERR_CUDA; }
    }
    if (!rc) rc = launch_tables(p, nullptr);
    if (!rc && p->logm >= 11 && p->logm <= 16) rc = init_iw3_tables(nullptr);
    if (!rc) {
        fill_kernel<<<(p->filt_stride + 255) / 256, 256>>>(p->filt_flat, p->filt_stride, (float)(1.0 / (2.0 * (double)n)));
        count_launch();
        rc = check_launch("fill_kernel");
    }
    if (!rc) {
        e = cudaStreamSynchronize(nullptr);
        if (e != cudaSuccess) { set_error("amplfi_plan_create: %s", cudaGetErrorString(e)); rc = AMPLFI_ERR_CUDA; }
    }
    if (rc) { amplfi_plan_destroy(p); return rc; }
    *out = p;
    return AMPLFI_OK;
}

int amplfi_plan_set_timing(amplfi_plan* p, int enable) {
    if (p == nullptr) { set_error("amplfi_plan_set_timing: null plan"); return AMPLFI_ERR_INVALID_ARG; }
    if (enable && p->ev_start[0] == nullptr) {
        for (int i = 0; i < AMPLFI_TIMING_RING; ++i) {
            if (cudaEventCreate(&p->ev_start[i]) != cudaSuccess || cudaEventCreate(&p->ev_stop[i]) != cudaSuccess) {
                set_error("amplfi_plan_set_timing: cudaEventCreate failed");
                return AMPLFI_ERR_CUDA;
            }
        }
    }
    p->timing = enable ? 1 : 0;
    p->ev_count = 0;
    return AMPLFI_OK;
}

int amplfi_plan_kernel_times(amplfi_plan* p, float* ms, int max) {
    if (p == nullptr || ms == nullptr) { set_error("amplfi_plan_kernel_times: null pointer"); return AMPLFI_ERR_INVALID_ARG; }
    int n = p->ev_count < max ? p->ev_count : max;
    for (int i = 0; i < n; ++i) {
        cudaError_t e = cudaEventSynchronize(p->ev_stop[i]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms[i], p->ev_start[i], p->ev_stop[i]);
        if (e != cudaSuccess) { set_error("amplfi_plan_kernel_times: %s", cudaGetErrorString(e)); return AMPLFI_ERR_CUDA; }
    }
    return n;
}

void amplfi_plan_destroy(amplfi_plan* p) {
    if (p == nullptr) return;
    if (p->ev_start[0] != nullptr)
        for (int i = 0; i < AMPLFI_TIMING_RING; ++i) { cudaEventDestroy(p->ev_start[i]); cudaEventDestroy(p->ev_stop[i]); }
    if (p->side) cudaStreamDestroy(p->side);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    cudaFree(p->tab_ci); cudaFree(p->tab_lnk); cudaFree(p->pd_table); cudaFree(p->coef); cudaFree(p->resp);
    cudaFree(p->resp2); cudaFree(p->filt_slots); cudaFree(p->filt_flat); cudaFree(p->fir_spec); cudaFree(p->fir_time);
    cudaFree(p->h0); cudaFree(p->filt); cudaFree(p->welch_part); cudaFree(p->d_det_ids); cudaFree(p->long_spec); cudaFree(p->long_filt_rows); cudaFree(p->long_h0_rows);
    delete p;
}

int amplfi_waveform_fd(const amplfi_plan* p, int approximant, int batch, const double* params, double f_lo,
                       double f_hi, float* hp, float* hc, int* flags, void* stream) {
    if (p == nullptr || params == nullptr || hp == nullptr || hc == nullptr) { set_error("amplfi_waveform_fd: null pointer"); return AMPLFI_ERR_INVALID_ARG; }
    if (batch < 1 || batch > p->max_batch) { set_error("amplfi_waveform_fd: batch %d outside [1, %d]", batch, p->max_batch); return AMPLFI_ERR_INVALID_ARG; }
    if (!known_approximant(approximant)) { set_error("amplfi_waveform_fd: unknown approximant %d", approximant); return AMPLFI_ERR_INVALID_ARG; }
    int rc = validate_band(p, f_lo, f_hi, "amplfi_waveform_fd");
    if (rc) return rc;
    if ((reinterpret_cast<size_t>(hp) | reinterpret_cast<size_t>(hc)) & 7) { set_error("amplfi_waveform_fd: hp/hc must be 8-byte aligned"); return AMPLFI_ERR_ALIGNMENT; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    rc = launch_prepare(p, approximant, batch, params, 0.0, f_lo, f_hi, 1.0, flags, st);
    if (rc) return rc;
    return launch_waveform_pol(p, batch, hp, hc, st);
}

int amplfi_project(const amplfi_plan* p, int batch, const double* params, double gmst, const float* hp,
                   const float* hc, float* h_det, double* resp, void* stream) {
    if (p == nullptr || params == nullptr) { set_error("amplfi_project: null pointer"); return AMPLFI_ERR_INVALID_ARG; }
    if (batch < 1 || batch > p->max_batch) { set_error("amplfi_project: batch %d outside [1, %d]", batch, p->max_batch); return AMPLFI_ERR_INVALID_ARG; }
    if (check_device(p, "amplfi_project")) return AMPLFI_ERR_INVALID_ARG;
    const bool any = hp != nullptr || hc != nullptr || h_det != nullptr;
    if (any && (hp == nullptr || hc == nullptr || h_det == nullptr)) { set_error("amplfi_project: hp, hc, h_det must be all given or all NULL"); return AMPLFI_ERR_INVALID_ARG; }
    if (!any && resp == nullptr) { set_error("amplfi_project: nothing to compute"); return AMPLFI_ERR_INVALID_ARG; }
    if (any && ((reinterpret_cast<size_t>(hp) | reinterpret_cast<size_t>(hc) | reinterpret_cast<size_t>(h_det)) & 7)) { set_error("amplfi_project: buffers must be 8-byte aligned"); return AMPLFI_ERR_ALIGNMENT; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = launch_prepare(p, -1, batch, params, gmst, 0.0, 0.0, 1.0, nullptr, st);
    if (rc) return rc;
    return launch_project(p, batch, hp, hc, h_det, resp, st);
}

int amplfi_psd_welch(const amplfi_plan* p, const float* bg, long n_bg, long row_stride, int noverlap, int detrend,
                     int average, float* psd, void* stream) {
    if (p == nullptr || bg == nullptr || psd == nullptr) { set_error("amplfi_psd_welch: null pointer"); return AMPLFI_ERR_INVALID_ARG; }
    if (p->nperseg == 0) { set_error("amplfi_psd_welch: plan was created with nperseg = 0"); return AMPLFI_ERR_INVALID_ARG; }
    if (check_device(p, "amplfi_psd_welch")) return AMPLFI_ERR_INVALID_ARG;
    if (n_bg < p->nperseg) { set_error("amplfi_psd_welch: nperseg %d > n_bg %ld", p->nperseg, n_bg); return AMPLFI_ERR_UNSUPPORTED_SIZE; }
    if (noverlap < 0 || noverlap >= p->nperseg || (detrend != 0 && detrend != 1) || (average != 0 && average != 1)) {
        set_error("amplfi_psd_welch: need 0 <= noverlap < nperseg, detrend in {0,1}, average in {0 mean, 1 median}");
        return AMPLFI_ERR_INVALID_ARG;
    }
    if (row_stride < n_bg) { set_error("amplfi_psd_welch: row_stride %ld < n_bg %ld", row_stride, n_bg); return AMPLFI_ERR_INVALID_ARG; }
    return launch_welch(p, bg, n_bg, row_stride, noverlap, detrend, average, psd, static_cast<cudaStream_t>(stream));
}

int amplfi_inject_whiten(const amplfi_plan* p, int batch, const float* noise, const long* offsets, long strip_len,
                         const float* h_det, int approximant, const double* params, double gmst, const float* psd,
                         int n_psd, double f_lo, double f_hi, float* out, void* stream) {
    if (p == nullptr || noise == nullptr || psd == nullptr || out == nullptr) { set_error("amplfi_inject_whiten: null pointer"); return AMPLFI_ERR_INVALID_ARG; }
    if (batch < 1 || batch > p->max_batch) { set_error("amplfi_inject_whiten: batch %d outside [1, %d]", batch, p->max_batch); return AMPLFI_ERR_INVALID_ARG; }
    int rc = validate_band(p, f_lo, f_hi, "amplfi_inject_whiten");
    if (rc) return rc;
    if (offsets != nullptr && strip_len < p->n) { set_error("amplfi_inject_whiten: strip_len %ld < n %d", strip_len, p->n); return AMPLFI_ERR_INVALID_ARG; }
    if (n_psd < 2 || ((p->n / 2) % (n_psd - 1)) != 0) { set_error("amplfi_inject_whiten: n_psd = %d does not divide the segment grid (n/2 = %d)", n_psd, p->n / 2); return AMPLFI_ERR_INVALID_ARG; }
    const bool fused = (h_det == nullptr && params != nullptr);
    if (fused && !known_approximant(approximant)) { set_error("amplfi_inject_whiten: unknown approximant %d", approximant); return AMPLFI_ERR_INVALID_ARG; }
    if ((reinterpret_cast<size_t>(out) & 7) || (reinterpret_cast<size_t>(noise) & 3) || (reinterpret_cast<size_t>(h_det) & 7)) { set_error("amplfi_inject_whiten: out/h_det must be 8-byte aligned, noise 4-byte aligned"); return AMPLFI_ERR_ALIGNMENT; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    rc = launch_filter(p, psd, n_psd, f_lo, f_hi, st);
    if (rc) return rc;
    if (fused) {
        rc = launch_prepare(p, approximant, batch, params, gmst, f_lo, f_hi, 2.0 * p->fs, nullptr, st);
        if (rc) return rc;
        rc = launch_waveform_h0(p, batch, st, v3_family(p));
        if (rc) return rc;
    }
    const bool timed = p->timing && p->ev_count < AMPLFI_TIMING_RING;
    if (timed) cudaEventRecord(p->ev_start[p->ev_count], st);
    rc = launch_inject_whiten(p, batch, noise, offsets, strip_len, h_det, fused ? 1 : 0, out, st);
    if (timed) { cudaEventRecord(p->ev_stop[p->ev_count], st); p->ev_count++; }
    return rc;
}

int amplfi_assemble_batch(const amplfi_plan* p, int batch, const float* bg, long n_bg, long row_stride, int noverlap,
                          int detrend, float* psd, const float* noise, const long* offsets, long strip_len,
                          int approximant, const double* params, double gmst, double f_lo, double f_hi, float* out,
                          void* stream) {
    if (p == nullptr || bg == nullptr || psd == nullptr || noise == nullptr || params == nullptr || out == nullptr) {
        set_error("amplfi_assemble_batch: null pointer");
        return AMPLFI_ERR_INVALID_ARG;
    }
    if (p->nperseg == 0) { set_error("amplfi_assemble_batch: plan was created with nperseg = 0"); return AMPLFI_ERR_INVALID_ARG; }
    if (batch < 1 || batch > p->max_batch) { set_error("amplfi_assemble_batch: batch %d outside [1, %d]", batch, p->max_batch); return AMPLFI_ERR_INVALID_ARG; }
    if (n_bg < p->nperseg) { set_error("amplfi_assemble_batch: nperseg %d > n_bg %ld", p->nperseg, n_bg); return AMPLFI_ERR_UNSUPPORTED_SIZE; }
    if (noverlap < 0 || noverlap >= p->nperseg || (detrend != 0 && detrend != 1)) { set_error("amplfi_assemble_batch: need 0 <= noverlap < nperseg, detrend in {0,1}"); return AMPLFI_ERR_INVALID_ARG; }
    if (row_stride < n_bg) { set_error("amplfi_assemble_batch: row_stride %ld < n_bg %ld", row_stride, n_bg); return AMPLFI_ERR_INVALID_ARG; }
    int rc = validate_band(p, f_lo, f_hi, "amplfi_assemble_batch");
    if (rc) return rc;
    if (offsets != nullptr && strip_len < p->n) { set_error("amplfi_assemble_batch: strip_len %ld < n %d", strip_len, p->n); return AMPLFI_ERR_INVALID_ARG; }
    if (!known_approximant(approximant)) { set_error("amplfi_assemble_batch: unknown approximant %d", approximant); return AMPLFI_ERR_INVALID_ARG; }
    if ((reinterpret_cast<size_t>(out) & 7) || (reinterpret_cast<size_t>(noise) & 3)) { set_error("amplfi_assemble_batch: out must be 8-byte aligned, noise 4-byte aligned"); return AMPLFI_ERR_ALIGNMENT; }
    const int n_psd = p->nperseg / 2 + 1;
    if (((p->n / 2) % (n_psd - 1)) != 0) { set_error("amplfi_assemble_batch: nperseg %d does not divide n %d", p->nperseg, p->n); return AMPLFI_ERR_INVALID_ARG; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const amplfi_plan* mp = p;
    // fork: PSD chain on the plan's stream, waveform chain on the caller's
    cudaError_t e = cudaEventRecord(mp->ev_fork, st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(mp->side, mp->ev_fork, 0);
    if (e != cudaSuccess) { set_error("amplfi_assemble_batch: fork: %s", cudaGetErrorString(e)); return AMPLFI_ERR_CUDA; }
    rc = launch_welch(p, bg, n_bg, row_stride, noverlap, detrend, 0, psd, mp->side);
    if (!rc) rc = launch_filter(p, psd, n_psd, f_lo, f_hi, mp->side);
    e = cudaEventRecord(mp->ev_join, mp->side);
    if (!rc) rc = launch_prepare(p, approximant, batch, params, gmst, f_lo, f_hi, 2.0 * p->fs, nullptr, st);
    if (!rc) rc = launch_waveform_h0(p, batch, st, v3_family(p));
    // join (always, so the side stream never runs past the call unobserved)
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, mp->ev_join, 0);
    if (e != cudaSuccess) { set_error("amplfi_assemble_batch: join: %s", cudaGetErrorString(e)); return AMPLFI_ERR_CUDA; }
    if (rc) return rc;
    const bool timed = p->timing && p->ev_count < AMPLFI_TIMING_RING;
    if (timed) cudaEventRecord(p->ev_start[p->ev_count], st);
    rc = launch_inject_whiten(p, batch, noise, offsets, strip_len, nullptr, 1, out, st);
    if (timed) { cudaEventRecord(p->ev_stop[p->ev_count], st); p->ev_count++; }
    return rc;
}

// shared validation of the inject/whiten family
static int validate_iw(const amplfi_plan* p, const char* who, int batch, const float* noise, const long* offsets, long strip_len,
                       const float* psd, int n_psd, double f_lo, double f_hi, const float* out) {
    if (p == nullptr || noise == nullptr || psd == nullptr || out == nullptr) { set_error("%s: null pointer", who); return AMPLFI_ERR_INVALID_ARG; }
    if (batch < 1 || batch > p->max_batch) { set_error("%s: batch %d outside [1, %d]", who, batch, p->max_batch); return AMPLFI_ERR_INVALID_ARG; }
    int rc = validate_band(p, f_lo, f_hi, who);
    if (rc) return rc;
    if (offsets != nullptr && strip_len < p->n) { set_error("%s: strip_len %ld < n %d", who, strip_len, p->n); return AMPLFI_ERR_INVALID_ARG; }
    if (n_psd < 2 || ((p->n / 2) % (n_psd - 1)) != 0) { set_error("%s: n_psd = %d does not divide the segment grid (n/2 = %d)", who, n_psd, p->n / 2); return AMPLFI_ERR_INVALID_ARG; }
    if ((reinterpret_cast<size_t>(out) & 7) || (reinterpret_cast<size_t>(noise) & 3)) { set_error("%s: out must be 8-byte aligned, noise 4-byte aligned", who); return AMPLFI_ERR_ALIGNMENT; }
    return AMPLFI_OK;
}

int amplfi_inject_whiten_views(const amplfi_plan* p, int batch, const float* noise, const long* offsets, long strip_len,
                               int approximant, const double* params, const double* t_shift, double gmst,
                               const float* psd, int n_psd, double f_lo, double f_hi, float* out, float* out2,
                               void* stream) {
    int rc = validate_iw(p, "amplfi_inject_whiten_views", batch, noise, offsets, strip_len, psd, n_psd, f_lo, f_hi, out);
    if (rc) return rc;
    if (params == nullptr || t_shift == nullptr || out2 == nullptr) { set_error("amplfi_inject_whiten_views: null pointer"); return AMPLFI_ERR_INVALID_ARG; }
    if (reinterpret_cast<size_t>(out2) & 7) { set_error("amplfi_inject_whiten_views: out2 must be 8-byte aligned"); return AMPLFI_ERR_ALIGNMENT; }
    if (!known_approximant(approximant)) { set_error("amplfi_inject_whiten_views: unknown approximant %d", approximant); return AMPLFI_ERR_INVALID_ARG; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    rc = launch_filter(p, psd, n_psd, f_lo, f_hi, st);
    if (!rc) rc = launch_prepare(p, approximant, batch, params, gmst, f_lo, f_hi, 2.0 * p->fs, nullptr, st);
    // n = 4096, 8192, 16384: one launch, one forward transform for both views (inject_whiten_v3.cu, VIEWS = 2)
    const bool one_launch = p->logm >= 11 && p->logm <= 13 && (reinterpret_cast<size_t>(out2) & 15) == 0;
    if (!rc) rc = launch_waveform_h0(p, batch, st, v3_family(p));
    // both views with the fp64-reduced phase, so that a zero shift reproduces the first view bit for bit
    IwOpts o;
    o.n_det = p->n_det; o.resp = nullptr; o.filt = nullptr; o.filt_stride = 0; o.crop = 0; o.phase64 = 1;
    o.out2 = nullptr; o.t_shift = nullptr;
    if (!rc && one_launch) {
        o.out2 = out2; o.t_shift = t_shift;
        return launch_inject_whiten(p, batch, noise, offsets, strip_len, nullptr, 1, out, st, &o);
    }
    if (!rc) rc = launch_shift_resp(p, batch, t_shift, st);
    if (!rc) rc = launch_inject_whiten(p, batch, noise, offsets, strip_len, nullptr, 1, out, st, &o);
    if (rc) return rc;
    o.resp = p->resp2;
    return launch_inject_whiten(p, batch, noise, offsets, strip_len, nullptr, 1, out2, st, &o);
}

int amplfi_waveform_td(const amplfi_plan* p, int approximant, int batch, const double* params, double f_lo, double f_hi,
                       float* h_t, int* flags, void* stream) {
    if (p == nullptr || params == nullptr || h_t == nullptr) { set_error("amplfi_waveform_td: null pointer"); return AMPLFI_ERR_INVALID_ARG; }
    if (batch < 1 || batch > p->max_batch) { set_error("amplfi_waveform_td: batch %d outside [1, %d]", batch, p->max_batch); return AMPLFI_ERR_INVALID_ARG; }
    if (!known_approximant(approximant)) { set_error("amplfi_waveform_td: unknown approximant %d", approximant); return AMPLFI_ERR_INVALID_ARG; }
    int rc = validate_band(p, f_lo, f_hi, "amplfi_waveform_td");
    if (rc) return rc;
    if (reinterpret_cast<size_t>(h_t) & 7) { set_error("amplfi_waveform_td: h_t must be 8-byte aligned"); return AMPLFI_ERR_ALIGNMENT; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    rc = launch_prepare(p, approximant, batch, params, 0.0, f_lo, f_hi, 2.0 * p->fs, flags, st);
    if (!rc) rc = launch_waveform_h0(p, batch, st, v3_family(p));
    if (!rc) rc = launch_td_resp(p, batch, st);
    if (rc) return rc;
    IwOpts o;
    o.n_det = 2; o.resp = p->resp2; o.filt = p->filt_flat; o.filt_stride = 0; o.crop = 0; o.phase64 = 0;
    o.out2 = nullptr; o.t_shift = nullptr;
    return launch_inject_whiten(p, batch, nullptr, nullptr, 0, nullptr, 1, h_t, st, &o);
}

int amplfi_inject_whiten_fir(const amplfi_plan* p, int batch, const float* noise, const long* offsets, long strip_len,
                             const float* h_det, int approximant, const double* params, double gmst, const float* psd,
                             int n_psd, double f_lo, double f_hi, double fduration, int crop, float* out, void* stream) {
    int rc = validate_iw(p, "amplfi_inject_whiten_fir", batch, noise, offsets, strip_len, psd, n_psd, f_lo, f_hi, out);
    if (rc) return rc;
    const long ntaps = llrint(fduration * p->fs);
    if (!(fduration > 0.0) || ntaps < 2 || ntaps > p->n || (ntaps & 3) || std::fabs((double)ntaps - fduration * p->fs) > 1e-6) {
        set_error("amplfi_inject_whiten_fir: fduration * fs must be a multiple of 4 in [4, n] (got %g s)", fduration);
        return AMPLFI_ERR_INVALID_ARG;
    }
    if (crop != 0 && crop != 1) { set_error("amplfi_inject_whiten_fir: crop must be 0 or 1"); return AMPLFI_ERR_INVALID_ARG; }
    if (crop && ntaps >= p->n) { set_error("amplfi_inject_whiten_fir: nothing left after cropping"); return AMPLFI_ERR_INVALID_ARG; }
    const bool fused = (h_det == nullptr && params != nullptr);
    if (fused && !known_approximant(approximant)) { set_error("amplfi_inject_whiten_fir: unknown approximant %d", approximant); return AMPLFI_ERR_INVALID_ARG; }
    if (reinterpret_cast<size_t>(h_det) & 7) { set_error("amplfi_inject_whiten_fir: h_det must be 8-byte aligned"); return AMPLFI_ERR_ALIGNMENT; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    rc = launch_filter(p, psd, n_psd, f_lo, f_hi, st);
    if (!rc) rc = launch_fir_truncate(p, fduration, st);
    if (!rc && fused) {
        rc = launch_prepare(p, approximant, batch, params, gmst, f_lo, f_hi, 2.0 * p->fs, nullptr, st);
        if (!rc) rc = launch_waveform_h0(p, batch, st, v3_family(p));
    }
    if (rc) return rc;
    IwOpts o;
    o.n_det = p->n_det; o.resp = nullptr; o.filt = nullptr; o.filt_stride = 0; o.crop = crop ? (int)(ntaps / 2) : 0; o.phase64 = 0;
    o.out2 = nullptr; o.t_shift = nullptr;
    return launch_inject_whiten(p, batch, noise, offsets, strip_len, h_det, fused ? 1 : 0, out, st, &o);
}

}  // extern "C"
