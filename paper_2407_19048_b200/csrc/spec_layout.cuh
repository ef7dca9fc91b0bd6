// spec_layout.cuh -- kernel-native ("slot") layout of the per-bin operands of the n = 16384 fused kernel.
//
// In inject_whiten_v3.cu thread t (0..255) and unit w (0..7) work on the two bin pairs (u = 2w)
//     lane 0:  k0 = t + 512 u      with partner M - k0,        lane 1:  k1 = t + 512 (u + 1)   with partner M - k1
// so the plan-internal operands (whitening filter, h0 of the fused path) are stored the way that thread reads them,
// 16 bytes per request, consecutive threads at consecutive addresses:
//     filter row [8][256] float4      = { f(k0), f(k1), f(M - k0), f(M - k1) }
//     h0 row     [2][8][256] float4   = first:  { re h(k0), re h(k1), im h(k0), im h(k1) },
//                                       second: { re h(M-k0), re h(M-k1), im h(M-k0), im h(M-k1) }
// Thread 0's second-type slots hold the self-paired bins 256 + 512 q (its lane-B butterfly).  Bins 0 .. M-1 each own
// exactly one slot; bin M (Nyquist) has none (the waveform is zero there, the filter is read from its linear row).
//
// h0 is produced only around the sample's band: a group of 32 consecutive threads (one warp of the consumer) writes its
// 32 slots of (second?, w) iff one of its two 32-bin windows overlaps [k_lo, k_hi] (bins outside the band written as
// exact zeros); the consumer skips exactly the other groups (window_needed() is the one rule both sides use).
#pragma once

namespace amplfi {
namespace slot {

constexpr int M = 8192, KL = 512;
constexpr int H0_ROW = 2 * 8 * 256 * 4;       // floats per sample (64 KB)
constexpr int FILT_ROW = 8 * 256 * 4;         // floats per detector (32 KB)

// bin k (0 <= k < M) -> (second, w, t, lane)
__host__ __device__ __forceinline__ void locate(int k, int& second, int& w, int& t, int& lane) {
    const int klow = k & (KL - 1), k3 = k >> 9;
    int u;
    if (klow < KL / 2) { second = 0; t = klow; u = k3; }
    else { second = 1; t = (KL - klow) & (KL / 2 - 1); u = 15 - k3; }
    w = u >> 1;
    lane = u & 1;
}
// float index of re h(k) in an h0 row (im at +2)
__host__ __device__ __forceinline__ int h0_index(int k) {
    int second, w, t, lane;
    locate(k, second, w, t, lane);
    return ((second * 8 + w) * 256 + t) * 4 + lane;
}
// float index of f(k) in a filter row
__host__ __device__ __forceinline__ int filt_index(int k) {
    int second, w, t, lane;
    locate(k, second, w, t, lane);
    return (w * 256 + t) * 4 + 2 * second + lane;
}
// bins of slot (second, w, t): lane 0 and lane 1
__host__ __device__ __forceinline__ void slot_bins(int second, int w, int t, int& kA, int& kB) {
    if (second == 0) { kA = t + KL * 2 * w; kB = kA + KL; }
    else if (t != 0) { kA = M - t - KL * 2 * w; kB = kA - KL; }
    else { kA = KL / 2 + KL * (15 - 2 * w); kB = kA - KL; }           // thread 0: bins 256 + 512 (15 - u)
}
// does warp `wi` (threads 32 wi .. 32 wi + 31) need the slots (second, w) for the band [k_lo, k_hi]?
// (for wi = 0 the windows are widened by thread 0's self-paired bins, which sit 256 away from the warp's other bins)
__host__ __device__ __forceinline__ bool window_needed(int second, int w, int wi, int k_lo, int k_hi) {
    const int base = 32 * wi + KL * 2 * w;
    int lo0, hi0;
    if (second == 0) { lo0 = base; hi0 = base + 31; }
    else { hi0 = M - base; lo0 = hi0 - 31; }
    const int lo1 = second == 0 ? lo0 + KL : lo0 - KL, hi1 = second == 0 ? hi0 + KL : hi0 - KL;
    bool need = (hi0 >= k_lo && lo0 <= k_hi) || (hi1 >= k_lo && lo1 <= k_hi);
    if (second == 1 && wi == 0) {
        const int s0 = KL / 2 + KL * (15 - 2 * w), s1 = s0 - KL;
        need = need || (s0 >= k_lo && s0 <= k_hi) || (s1 >= k_lo && s1 <= k_hi);
    }
    return need;
}

}  // namespace slot
}  // namespace amplfi
