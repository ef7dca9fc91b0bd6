// amplfi_internal.h -- plan layout and launch entry points shared by the library's translation units.
#pragma once
#include <cuda_runtime.h>

#include <atomic>

#include "../../include/amplfi.h"
#include "phenomd_table.h"

#define AMPLFI_TIMING_RING 512
#define AMPLFI_QNM_NODES 512         /* Kerr (2,2,0) mode on a grid uniform in sqrt(1 - a/M), a/M from +0.998 down to -0.998 */
#define AMPLFI_QNM_OFFSET 216        /* doubles: the mode table follows the 19 x 11 fit table in plan->pd_table */

namespace amplfi {
struct WfCoef;
struct DetResp;
}

struct amplfi_plan {
    int n;                 // samples per segment
    int n_bins;            // n/2 + 1
    int logm;              // log2(n/2)
    double fs, t_seg;
    int n_det;
    int det_ids[3];
    int max_batch;
    int nperseg;           // 0: no Welch
    mutable int last_approx;       // approximant of the last launch_prepare (the waveform launch that follows evaluates that family)
    int device;
    int sm_count;
    // device tables / workspace (owned)
    double* tab_ci;        // [n_bins] k^(-1/3)   (tab_ci[0] = 0)
    double* tab_lnk;       // [n_bins] ln k       (tab_lnk[0] = 0)
    double* pd_table;      // [19*11] fit table, then at AMPLFI_QNM_OFFSET the Kerr mode table [AMPLFI_QNM_NODES][2]
    amplfi::WfCoef* coef;  // [max_batch]
    amplfi::DetResp* resp; // [max_batch * n_det]
    amplfi::DetResp* resp2; // [max_batch * 3]  second view: resp with dt + t_shift[b]; also the two "polarisation detectors" of
                           //                  amplfi_waveform_td ((F+, Fx, dt) = (1,0,0), (0,1,0) per sample)
    float2* h0;            // [max_batch * n_bins]   fused path: 2 fs h0
    float* filt;           // [n_det * filt_stride]  whitening filter incl. 1/(2n); rows padded to 16 B
    float* filt_slots;     // n = 4096 .. 131072: the same filter in the slot layout of the fused kernel [n_det * n/2] (spec_layout.cuh)
    int filt_stride;       // n_bins rounded up to a multiple of 4
    float* filt_flat;      // [filt_stride] constant 1/(2n): the "no filter" row of the inverse-only launches
    float2* fir_spec;      // [n_det * n_bins]  truncated-filter construction: spectrum-side workspace
    float* fir_time;       // [n_det * n]       truncated-filter construction: time-side workspace
    float* welch_part;     // [n_det * max_seg * (nperseg/2+1)]
    int welch_max_seg;
    int* d_det_ids;        // [3]
    float2* long_spec;     // n >= 2^18: rows of one chunk of units [long_chunk, n/32768 + 1, 16384] (L2-resident)
    int long_chunk;        // units per chunk
    float* long_filt_rows; // n >= 2^18: the filter in the [c][e] row layout of inject_whiten_long.cu [n_det, n/32768 + 1, 16384]
    float2* long_h0_rows;  // ... and the fused path's h0 [max_batch, n/32768 + 1, 16384]
    // amplfi_assemble_batch: PSD chain runs on `side`, forked from / joined into the caller's stream
    cudaStream_t side;
    cudaEvent_t ev_fork, ev_join;
    // optional device timing of the dominant kernel (amplfi_plan_set_timing)
    // (mutable: the compute calls take a const plan; a plan is used by one host thread and one stream at a time)
    int timing;
    mutable int ev_count;
    cudaEvent_t ev_start[AMPLFI_TIMING_RING], ev_stop[AMPLFI_TIMING_RING];
};

namespace amplfi {

void set_error(const char* fmt, ...);
int check_launch(const char* what);
void count_launch(int n = 1);

// Opt a kernel in to `bytes` of dynamic shared memory once per device (the attribute is per device; setting it twice is
// harmless, so a racing second thread costs one redundant call).  `done` is a per-kernel bit mask of devices.
template <class Kernel>
inline int ensure_dynamic_smem(Kernel kernel, int bytes, std::atomic<unsigned>& done) {
    int dev = 0;
    cudaGetDevice(&dev);
    const unsigned bit = 1u << (dev & 31);
    if (done.load(std::memory_order_acquire) & bit) return AMPLFI_OK;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) { set_error("cudaFuncSetAttribute: %s", cudaGetErrorString(e)); return AMPLFI_ERR_CUDA; }
    done.fetch_or(bit, std::memory_order_release);
    return AMPLFI_OK;
}

// kerr_qnm.cu (host): (Re M omega, -Im M omega) of the Kerr (2,2,0) mode per node, computed once per process; nullptr on failure
const double* kerr_qnm_table();

// waveform.cu
int launch_prepare(const amplfi_plan* p, int approximant, int batch, const double* params, double gmst,
                   double f_lo, double f_hi, double amp_mul, int* flags, cudaStream_t st);
int launch_waveform_pol(const amplfi_plan* p, int batch, float* hp, float* hc, cudaStream_t st);
int launch_waveform_h0(const amplfi_plan* p, int batch, cudaStream_t st, int slots);   // slots: spec_layout.cuh (n = 4096 .. 131072)
int launch_project(const amplfi_plan* p, int batch, const float* hp, const float* hc, float* h_det,
                   double* resp_out, cudaStream_t st);
int launch_tables(amplfi_plan* p, cudaStream_t st);

// welch.cu
int launch_welch(const amplfi_plan* p, const float* bg, long n_bg, long row_stride, int noverlap, int detrend, int average,
                 float* psd, cudaStream_t st);

enum { MODE_NONE = 0, MODE_HDET = 1, MODE_FUSED = 2 };

struct IwArgs {
    const float* noise;       // dense [B, D, N] or strip [D, L]; nullptr: no data, the spectrum starts at zero and the
                              // forward transform is skipped (inverse-only launches: time-domain waveform, filter design)
    const long* offsets;      // nullptr: dense
    long strip_len;
    const float2* h_det;      // MODE_HDET: [B, D, K]
    const float2* h0;         // MODE_FUSED: [B, K] (2 fs h0)
    const WfCoef* coef;
    const DetResp* resp;
    const float* filt;        // [D, filt_stride]
    int filt_stride;
    const float* filt_slots;  // n = 16384: [D, 8192] slot layout (stride 0 when filt_stride is 0); h0 is then in slot layout too
    float* out;               // [B, D, N - 2 crop]
    float* out2;              // packed kernel, two-view launch: second view [B, D, N] (16-byte aligned); else nullptr
    const double* t_shift;    // two-view launch: [B] seconds added to the arrival time in the second view
    int crop;                 // samples dropped at each end of every output row (even)
    int phase64;              // packed kernel: reduce the projection phase in fp64 (needed when |dt| can reach ~1 s)
    int n_det;
    float two_fs;
    float inv_tseg;
    int prefetch_ahead;       // units ahead whose noise segment is prefetched into L2 (packed kernel)
};

// optional overrides of launch_inject_whiten (defaults: the plan's detectors, responses and filter, no crop)
struct IwOpts {
    int n_det;                // units per sample (2 for the polarisations of amplfi_waveform_td, 1 for filter design)
    const DetResp* resp;      // nullptr: plan->resp
    const float* filt;        // nullptr: plan->filt (a given row must be constant: it is also used as its own slot layout)
    int filt_stride;
    int crop;
    int phase64;
    float* out2;              // with t_shift: both views in one launch (n = 16384 only)
    const double* t_shift;
};


// inject_whiten_v3.cu (three-pass cosine-tangent kernel for n = 4096, 8192, 16384)
int launch_iw3(const IwArgs& a, int logm /*11 .. 14*/, int mode, int units, cudaStream_t st);
int init_iw3_tables(cudaStream_t st);

// inject_whiten.cu
int launch_filter(const amplfi_plan* p, const float* psd, int n_psd, double f_lo, double f_hi, cudaStream_t st);
int launch_inject_whiten(const amplfi_plan* p, int batch, const float* noise, const long* offsets,
                         long strip_len, const float* h_det, int fused, float* out, cudaStream_t st,
                         const IwOpts* opts = nullptr);
int launch_fir_truncate(const amplfi_plan* p, double fduration, cudaStream_t st);
int launch_shift_resp(const amplfi_plan* p, int batch, const double* t_shift, cudaStream_t st);
int launch_td_resp(const amplfi_plan* p, int batch, cudaStream_t st);
int setup_inject_whiten_attrs();

// inject_whiten_long.cu (n = 2^18 .. 2^20: four-step transform around rows of 16384 complex points)
size_t long_scratch_floats2(int chunk_units, int rdec);
size_t long_row_elems(int rdec);
int launch_inject_whiten_long(const amplfi_plan* p, const IwArgs& a, int mode, int units, cudaStream_t st);

}  // namespace amplfi
