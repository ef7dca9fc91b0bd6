// welch.cu -- segmented Welch PSD: detrend, Hann window, real FFT, |X|^2 in one pass per segment, then
// a fixed-order mean over segments (deterministic; no atomics).
// PAPER.md:101 "power spectra estimation ... carried out on the GPU"; "The power spectra is
// fit to this background chunk".  Estimator parameters: BASELINE.json configs (Hann, 50 % overlap, mean).
#include "amplfi_internal.h"
#include "fft_core.cuh"

namespace amplfi {

constexpr float kStrainScale = 1180591620717411303424.0f;   // 2^70: strain -> O(1); |X|^2 then carries 2^140

// One CTA per (detector, segment).  part[d][seg][k] = |FFT(w (x - mean))[k]|^2 (scaled by 2^140).
template <int LOGM>
__global__ void __launch_bounds__(Fft<LOGM>::T) welch_segment_kernel(const float* __restrict__ bg, long row_stride, int step,
                                                                     int nseg, int detrend, float* __restrict__ part) {
    using F = Fft<LOGM>;
    constexpr int M = F::M, NPS = 2 * M, RA = F::RA, RC = F::RC, T = F::T, LB = F::LB;
    extern __shared__ float2 sm[];
    __shared__ float red[32];
    const int seg = blockIdx.x, d = blockIdx.y, tid = threadIdx.x;
    const float* x = bg + (size_t)d * row_stride + (size_t)seg * step;

    float2 v[F::NA][RA];
    float sum = 0.f;
#pragma unroll
    for (int a = 0; a < F::NA; ++a) {
        const int jA = tid + a * T;
#pragma unroll
        for (int nA = 0; nA < RA; ++nA) {
            const int m = nA * LB + jA;
            float2 z = make_float2(x[2 * m] * kStrainScale, x[2 * m + 1] * kStrainScale);
            v[a][nA] = z;
            sum += z.x + z.y;
        }
    }
    float mean = 0.f;
    if (detrend) {
        // fixed-order block reduction: warp shuffles, then warp 0 over the per-warp sums
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if ((tid & 31) == 0) red[tid >> 5] = sum;
        __syncthreads();
        float tot = 0.f;
        for (int w = 0; w < (T + 31) / 32; ++w) tot += red[w];
        mean = tot * (1.0f / (float)NPS);
    }
#pragma unroll
    for (int a = 0; a < F::NA; ++a) {
        const int jA = tid + a * T;
#pragma unroll
        for (int nA = 0; nA < RA; ++nA) {
            const int m = nA * LB + jA;
            // periodic Hann at samples 2m, 2m+1: w[n] = (1 - cos(2 pi n / NPS)) / 2
            const float w0 = 0.5f - 0.5f * cospif((float)(2 * m) * (2.0f / (float)NPS));
            const float w1 = 0.5f - 0.5f * cospif((float)(2 * m + 1) * (2.0f / (float)NPS));
            v[a][nA].x = (v[a][nA].x - mean) * w0;
            v[a][nA].y = (v[a][nA].y - mean) * w1;
        }
        F::pass_a_fwd(v[a], jA, sm);
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < F::NB; ++i) F::pass_b_fwd(tid + i * T, sm);
    __syncthreads();
    int klow_a, klow_b;
    pass_c_klow<LOGM>(tid, klow_a, klow_b);
    float2 va[RC], vb[RC];
    F::pass_c_fwd(klow_a, va, sm);
    F::pass_c_fwd(klow_b, vb, sm);

    float* out = part + ((size_t)d * nseg + seg) * (M + 1);
    for_each_bin_pair<LOGM>(
        tid, va, vb,
        [&](int k, float2& za, float2& zb) {
            float2 xa, xb;
            split_pair(za, zb, twiddle<2 * M>(k), xa, xb);
            out[k] = 0.25f * (xa.x * xa.x + xa.y * xa.y);
            out[M - k] = 0.25f * (xb.x * xb.x + xb.y * xb.y);
        },
        [&](int k, float2& z) {
            float2 xa, xb;
            split_pair(z, z, twiddle<2 * M>(k), xa, xb);
            out[k] = 0.25f * (xa.x * xa.x + xa.y * xa.y);
        },
        [&](float2& z) {
            const float dc = z.x + z.y, ny = z.x - z.y;
            out[0] = dc * dc;
            out[M] = ny * ny;
        });
}

// psd[d][k] = c_k * (sum_seg part) / (nseg * fs * sum w^2), c_k = 2 except DC/Nyquist; sum w^2 = 3 NPS / 8.
// Fixed summation order (deterministic): warp j of a CTA sums the segments s = j, j + 8, ... of 32 bins (coalesced 128-byte
// rows, at most ceil(nseg / 8) dependent loads instead of nseg), then the eight partial sums are added in the order j = 0..7.
constexpr int MEAN_PARTS = 8;
__global__ void __launch_bounds__(32 * MEAN_PARTS) welch_mean_kernel(const float* __restrict__ part, int nseg, int n_w,
                                                                     float scale, float* __restrict__ psd, int accumulate) {
    __shared__ float partial[MEAN_PARTS][32];
    const int lane = threadIdx.x & 31, j = threadIdx.x >> 5;
    const int k = blockIdx.x * 32 + lane;
    const int d = blockIdx.y;
    float acc = 0.f;
    if (k < n_w) {
        const float* p = part + (size_t)d * nseg * n_w + k;
        for (int s = j; s < nseg; s += MEAN_PARTS) acc += p[(size_t)s * n_w];
    }
    partial[j][lane] = acc;
    __syncthreads();
    if (j == 0 && k < n_w) {
        float tot = partial[0][lane];
#pragma unroll
        for (int q = 1; q < MEAN_PARTS; ++q) tot += partial[q][lane];
        const float ck = (k == 0 || k == n_w - 1) ? 1.0f : 2.0f;
        // (accumulate: a later group of segments of a long background, added in launch order)
        psd[(size_t)d * n_w + k] = accumulate ? psd[(size_t)d * n_w + k] + tot * scale * ck : tot * scale * ck;
    }
}

// Median over segments: per bin, the middle order statistic of the nseg periodogram values (the
// mean of the two middle ones for even nseg), found by rank counting over a shared-memory column (nseg <= 256, so the
// O(nseg^2) comparisons are a few thousand per bin); ties are broken by segment index, so ranks are a permutation and
// exactly one candidate has each of the two middle ranks.  A CTA serves 64 bins with MED_PARTS threads per bin, each
// ranking every MED_PARTS-th candidate.  `scale` carries 1 / (median_bias(nseg) fs sum w^2).
constexpr int MED_PARTS = 8;
__global__ void __launch_bounds__(64 * MED_PARTS) welch_median_kernel(const float* __restrict__ part, int nseg, int n_w,
                                                                      float scale, float* __restrict__ psd) {
    extern __shared__ float col[];                       // [nseg][64], then the two middle values [2][64]
    const int lane = threadIdx.x & 63, sub = threadIdx.x >> 6;
    const int k = blockIdx.x * 64 + lane;
    const int d = blockIdx.y;
    const bool live = k < n_w;
    float* mid = col + nseg * 64;
    if (live) {
        const float* p = part + (size_t)d * nseg * n_w + k;
        for (int s = sub; s < nseg; s += MED_PARTS) col[s * 64 + lane] = p[(size_t)s * n_w];
    }
    __syncthreads();
    if (live) {
        const int r_lo = (nseg - 1) >> 1, r_hi = nseg >> 1;   // equal for odd nseg
        for (int i = sub; i < nseg; i += MED_PARTS) {
            const float vi = col[i * 64 + lane];
            int rank = 0;
            for (int j = 0; j < nseg; ++j) {
                const float vj = col[j * 64 + lane];
                rank += (vj < vi || (vj == vi && j < i)) ? 1 : 0;
            }
            if (rank == r_lo) mid[lane] = vi;
            if (rank == r_hi) mid[64 + lane] = vi;
        }
    }
    __syncthreads();
    if (live && sub == 0) {
        const float ck = (k == 0 || k == n_w - 1) ? 1.0f : 2.0f;
        psd[(size_t)d * n_w + k] = 0.5f * (mid[lane] + mid[64 + lane]) * scale * ck;
    }
}

template <int LOGM>
static int launch_welch_t(const amplfi_plan* p, const float* bg, long row_stride, int step, int nseg, int detrend,
                          cudaStream_t st) {
    using F = Fft<LOGM>;
    static std::atomic<unsigned> attr_done{0};
    const int arc = ensure_dynamic_smem(welch_segment_kernel<LOGM>, (int)F::SMEM_BYTES, attr_done);
    if (arc) return arc;
    dim3 grid(nseg, p->n_det);
    welch_segment_kernel<LOGM><<<grid, F::T, F::SMEM_BYTES, st>>>(bg, row_stride, step, nseg, detrend, p->welch_part);
    count_launch();
    return check_launch("welch_segment_kernel");
}

// E[median] / E[mean] of nseg exponentially distributed periodogram values: the k-th smallest of n unit exponentials has
// expectation sum_{j = n-k+1}^{n} 1/j (host arithmetic on a launch parameter, like the mean's 1/nseg).
static double median_bias(int n) {
    auto e_order = [n](int k) { double s = 0.0; for (int j = n - k + 1; j <= n; ++j) s += 1.0 / (double)j; return s; };
    return (n & 1) ? e_order((n + 1) / 2) : 0.5 * (e_order(n / 2) + e_order(n / 2 + 1));
}

int launch_welch(const amplfi_plan* p, const float* bg, long n_bg, long row_stride, int noverlap, int detrend, int average,
                 float* psd, cudaStream_t st) {
    const int nps = p->nperseg;
    const int step = nps - noverlap;
    const long nseg_l = (n_bg - nps) / step + 1;
    const int n_w = nps / 2 + 1;
    auto segments = [&](const float* base, int nseg) {
        switch (ilog2(nps) - 1) {
            case 9: return launch_welch_t<9>(p, base, row_stride, step, nseg, detrend, st);
            case 10: return launch_welch_t<10>(p, base, row_stride, step, nseg, detrend, st);
            case 11: return launch_welch_t<11>(p, base, row_stride, step, nseg, detrend, st);
            case 12: return launch_welch_t<12>(p, base, row_stride, step, nseg, detrend, st);
            case 13: return launch_welch_t<13>(p, base, row_stride, step, nseg, detrend, st);
            case 14: return launch_welch_t<14>(p, base, row_stride, step, nseg, detrend, st);
            default: set_error("amplfi_psd_welch: unsupported nperseg %d", nps); return (int)AMPLFI_ERR_UNSUPPORTED_SIZE;
        }
    };
    if (nseg_l > p->welch_max_seg) {
        // A long background (the PSD is fit to the whole resident chunk, ~20 000 two-second segments for a
        // quarter day): groups of welch_max_seg segments, their sums added to psd in launch order (still deterministic).
        if (average == 1) {
            set_error("amplfi_psd_welch: the median needs all %ld segments at once, the plan's workspace holds %d", nseg_l,
                      p->welch_max_seg);
            return AMPLFI_ERR_UNSUPPORTED_SIZE;
        }
        const float gscale = (float)(1.0 / ((double)nseg_l * p->fs * 0.375 * (double)nps));
        dim3 ggrid((n_w + 31) / 32, p->n_det);
        for (long s0 = 0; s0 < nseg_l; s0 += p->welch_max_seg) {
            const int ng = (int)(nseg_l - s0 < p->welch_max_seg ? nseg_l - s0 : p->welch_max_seg);
            const int grc = segments(bg + s0 * step, ng);
            if (grc) return grc;
            welch_mean_kernel<<<ggrid, 32 * MEAN_PARTS, 0, st>>>(p->welch_part, ng, n_w, gscale, psd, s0 != 0);
            count_launch();
        }
        return check_launch("welch_mean_kernel");
    }
    const int nseg = (int)nseg_l;
    const int rc = segments(bg, nseg);
    if (rc) return rc;
    if (average == 1) {
        static std::atomic<unsigned> attr_done{0};
        const int arc = ensure_dynamic_smem(welch_median_kernel, (256 + 2) * 64 * (int)sizeof(float), attr_done);
        if (arc) return arc;
        const float mscale = (float)(1.0 / (median_bias(nseg) * p->fs * 0.375 * (double)nps));
        dim3 mgrid((n_w + 63) / 64, p->n_det);
        welch_median_kernel<<<mgrid, 64 * MED_PARTS, (size_t)(nseg + 2) * 64 * sizeof(float), st>>>(p->welch_part, nseg, n_w, mscale, psd);
        count_launch();
        return check_launch("welch_median_kernel");
    }
    const float scale = (float)(1.0 / ((double)nseg * p->fs * 0.375 * (double)nps));
    dim3 grid((n_w + 31) / 32, p->n_det);
    welch_mean_kernel<<<grid, 32 * MEAN_PARTS, 0, st>>>(p->welch_part, nseg, n_w, scale, psd, 0);
    count_launch();
    return check_launch("welch_mean_kernel");
}

}  // namespace amplfi

// ---------------------------------------------------------------------------------------------------------------------
// amplfi_psd_welch_noalloc: the Welch estimate for callers that may not allocate device memory (code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc).  The same two kernels as amplfi_psd_welch, but no plan:
// the per-segment periodograms go to a file-scope device array instead of the plan's workspace.
//   - AMPLFI_NOALLOC_WELCH_FLOATS floats (4 MiB), held by every GPU that loads the library until the process exits;
//   - shared by all calls: calls that overlap on the GPU (different streams, different threads) race on it;
//   - nothing in it has to start at zero: welch_segment_kernel overwrites every value welch_mean_kernel reads, so what
//     the previous call left behind is never seen.
// In host code the array's name is only a stand-in; the device address comes from cudaGetSymbolAddress, taken once per
// device with that device current, and is what the kernels are given.
namespace amplfi {
namespace {

static __device__ __align__(256) float g_welch_scratch[AMPLFI_NOALLOC_WELCH_FLOATS];

constexpr int kMaxDevices = 64;
float* g_scratch_ptr[kMaxDevices];
std::atomic<int> g_scratch_ready[kMaxDevices];

// device address of g_welch_scratch on the current device (resolved at the first call on that device)
int noalloc_scratch(float** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { set_error("amplfi_psd_welch_noalloc: cudaGetDevice: %s", cudaGetErrorString(e)); return AMPLFI_ERR_CUDA; }
    if (dev < 0 || dev >= kMaxDevices) { set_error("amplfi_psd_welch_noalloc: device ordinal %d not supported", dev); return AMPLFI_ERR_INVALID_ARG; }
    if (!g_scratch_ready[dev].load(std::memory_order_acquire)) {
        float* q = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&q), g_welch_scratch);
        if (e != cudaSuccess || q == nullptr) {
            set_error("amplfi_psd_welch_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return AMPLFI_ERR_CUDA;
        }
        g_scratch_ptr[dev] = q;
        g_scratch_ready[dev].store(1, std::memory_order_release);
    }
    *out = g_scratch_ptr[dev];
    return AMPLFI_OK;
}

template <int LOGM>
int noalloc_segments_t(const float* bg, long row_stride, int step, int nseg, int detrend, int n_det, float* part, cudaStream_t st) {
    using F = Fft<LOGM>;
    static std::atomic<unsigned> attr_done{0};
    const int arc = ensure_dynamic_smem(welch_segment_kernel<LOGM>, (int)F::SMEM_BYTES, attr_done);
    if (arc) return arc;
    dim3 grid(nseg, n_det);
    welch_segment_kernel<LOGM><<<grid, F::T, F::SMEM_BYTES, st>>>(bg, row_stride, step, nseg, detrend, part);
    count_launch();
    return check_launch("welch_segment_kernel");
}

}  // namespace
}  // namespace amplfi

extern "C" int amplfi_psd_welch_noalloc(const float* bg, long n_bg, long row_stride, int n_det, double fs, int nperseg,
                                        int noverlap, int detrend, float* psd, void* stream) {
    using namespace amplfi;
    const char* who = "amplfi_psd_welch_noalloc";
    if (bg == nullptr || psd == nullptr) { set_error("%s: null pointer", who); return AMPLFI_ERR_INVALID_ARG; }
    if (n_det < 1 || n_det > 3 || !(fs > 0.0)) { set_error("%s: need 1 <= n_det <= 3 and fs > 0", who); return AMPLFI_ERR_INVALID_ARG; }
    if (nperseg < 1024 || nperseg > 32768 || (nperseg & (nperseg - 1)) != 0) {
        set_error("%s: nperseg %d is not a power of two in [2^10, 2^15]", who, nperseg);
        return AMPLFI_ERR_UNSUPPORTED_SIZE;
    }
    if (n_bg < nperseg) { set_error("%s: nperseg %d > n_bg %ld", who, nperseg, n_bg); return AMPLFI_ERR_UNSUPPORTED_SIZE; }
    if (noverlap < 0 || noverlap >= nperseg || (detrend != 0 && detrend != 1)) {
        set_error("%s: need 0 <= noverlap < nperseg, detrend in {0,1}", who);
        return AMPLFI_ERR_INVALID_ARG;
    }
    if (row_stride < n_bg) { set_error("%s: row_stride %ld < n_bg %ld", who, row_stride, n_bg); return AMPLFI_ERR_INVALID_ARG; }
    const int step = nperseg - noverlap, n_w = nperseg / 2 + 1;
    const long nseg_l = (n_bg - nperseg) / step + 1;
    const long need = (long)n_det * nseg_l * n_w;
    if (need > (long)AMPLFI_NOALLOC_WELCH_FLOATS) {
        set_error("%s: n_det %d x %ld segments x %d bins = %ld floats of scratch, the static array holds %ld "
                  "(use amplfi_psd_welch with a plan for larger backgrounds)", who, n_det, nseg_l, n_w, need,
                  (long)AMPLFI_NOALLOC_WELCH_FLOATS);
        return AMPLFI_ERR_UNSUPPORTED_SIZE;
    }
    float* part = nullptr;
    int rc = noalloc_scratch(&part);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int nseg = (int)nseg_l;
    switch (ilog2(nperseg) - 1) {
        case 9: rc = noalloc_segments_t<9>(bg, row_stride, step, nseg, detrend, n_det, part, st); break;
        case 10: rc = noalloc_segments_t<10>(bg, row_stride, step, nseg, detrend, n_det, part, st); break;
        case 11: rc = noalloc_segments_t<11>(bg, row_stride, step, nseg, detrend, n_det, part, st); break;
        case 12: rc = noalloc_segments_t<12>(bg, row_stride, step, nseg, detrend, n_det, part, st); break;
        case 13: rc = noalloc_segments_t<13>(bg, row_stride, step, nseg, detrend, n_det, part, st); break;
        default: rc = noalloc_segments_t<14>(bg, row_stride, step, nseg, detrend, n_det, part, st); break;
    }
    if (rc) return rc;
    const float scale = (float)(1.0 / ((double)nseg * fs * 0.375 * (double)nperseg));
    dim3 grid((n_w + 31) / 32, n_det);
    welch_mean_kernel<<<grid, 32 * MEAN_PARTS, 0, st>>>(part, nseg, n_w, scale, psd, 0);
    count_launch();
    return check_launch("welch_mean_kernel");
}
