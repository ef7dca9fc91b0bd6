// spec_layout.cuh -- kernel-native ("slot") layout of the per-bin operands of the three-pass fused kernel
// (inject_whiten_v3.cu: n = 4096 ... 131072, i.e. M = n/2 = 2048 ... 65536 complex points).
//
// With KL = M/16 and T = KL/2 threads, thread t (0 .. T-1) and unit w (0..7) work on the two bin pairs (u = 2w)
//     lane 0:  k0 = t + KL u      with partner M - k0,        lane 1:  k1 = t + KL (u + 1)   with partner M - k1
// so the plan-internal operands (whitening filter, h0 of the fused path) are stored the way that thread reads them,
// 16 bytes per request, consecutive threads at consecutive addresses:
//     filter row [8][T] float4      = { f(k0), f(k1), f(M - k0), f(M - k1) }                               (M floats)
//     h0 row     [2][8][T] float4   = first:  { re h(k0), re h(k1), im h(k0), im h(k1) },                   (2M floats)
//                                     second: { re h(M-k0), re h(M-k1), im h(M-k0), im h(M-k1) }
// Thread 0's second-type slots hold the self-paired bins KL/2 + KL q (its lane-B butterfly).  Bins 0 .. M-1 each own
// exactly one slot; bin M (Nyquist) has none (the waveform is zero there, the filter is read from its linear row).
//
// h0 is produced only around the sample's band: a group of 32 consecutive threads (one warp of the consumer) writes its
// 32 slots of (second?, w) iff one of its two 32-bin windows overlaps [k_lo, k_hi] (bins outside the band written as
// exact zeros); the consumer skips exactly the other groups (window_needed() is the one rule both sides use).
#pragma once

namespace amplfi {
namespace slot {

// geometry of a segment length: kl = M / 16 (128 ... 4096), T = kl / 2 threads, M = 16 kl
__host__ __device__ __forceinline__ int h0_row(int kl) { return 32 * kl; }        // floats per sample (2M)
__host__ __device__ __forceinline__ int filt_row(int kl) { return 16 * kl; }      // floats per detector (M)

// bin k (0 <= k < M) -> (second, w, t, lane)
__host__ __device__ __forceinline__ void locate(int kl, int k, int& second, int& w, int& t, int& lane) {
    const int klow = k & (kl - 1), k3 = k / kl;
    int u;
    if (klow < kl / 2) { second = 0; t = klow; u = k3; }
    else { second = 1; t = (kl - klow) & (kl / 2 - 1); u = 15 - k3; }
    w = u >> 1;
    lane = u & 1;
}
// float index of re h(k) in an h0 row (im at +2)
__host__ __device__ __forceinline__ int h0_index(int kl, int k) {
    int second, w, t, lane;
    locate(kl, k, second, w, t, lane);
    return ((second * 8 + w) * (kl / 2) + t) * 4 + lane;
}
// float index of f(k) in a filter row
__host__ __device__ __forceinline__ int filt_index(int kl, int k) {
    int second, w, t, lane;
    locate(kl, k, second, w, t, lane);
    return (w * (kl / 2) + t) * 4 + 2 * second + lane;
}
// bins of slot (second, w, t): lane 0 and lane 1
__host__ __device__ __forceinline__ void slot_bins(int kl, int second, int w, int t, int& kA, int& kB) {
    // first: (t + kl 2w, + kl);  second: (M - t - kl 2w, - kl), thread 0: the self-paired bins kl/2 + kl (15 - 2w), - kl
    // (branch-free: the producer kernel evaluates this once per slot group)
    const int base = kl * 2 * w;
    const int tt = t != 0 ? t : kl / 2;
    kA = second ? 16 * kl - base - tt : base + t;
    kB = second ? kA - kl : kA + kl;
}
// does warp `wi` (threads 32 wi .. 32 wi + 31) need the slots (second, w) for the band [k_lo, k_hi]?
// (for wi = 0 the windows are widened by thread 0's self-paired bins, which sit KL/2 away from the warp's other bins)
__host__ __device__ __forceinline__ bool window_needed(int kl, int second, int w, int wi, int k_lo, int k_hi) {
    const int m = 16 * kl;
    const int base = 32 * wi + kl * 2 * w;
    int lo0, hi0;
    if (second == 0) { lo0 = base; hi0 = base + 31; }
    else { hi0 = m - base; lo0 = hi0 - 31; }
    const int lo1 = second == 0 ? lo0 + kl : lo0 - kl, hi1 = second == 0 ? hi0 + kl : hi0 - kl;
    bool need = (hi0 >= k_lo && lo0 <= k_hi) || (hi1 >= k_lo && lo1 <= k_hi);
    if (second == 1 && wi == 0) {
        const int s0 = kl / 2 + kl * (15 - 2 * w), s1 = s0 - kl;
        need = need || (s0 >= k_lo && s0 <= k_hi) || (s1 >= k_lo && s1 <= k_hi);
    }
    return need;
}

}  // namespace slot
}  // namespace amplfi
