"""Seeded synthetic inputs for the five BASELINE.json configs (c0..c4).

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench, and therefore
holds none of the method's arithmetic: only random draws from the paper's priors (Table 1,
PAPER.md:130-141), the analytic noise curve BASELINE.json gives for its configs, and the
colouring of Gaussian noise with it (numpy.fft, an input synthesis step, not the method's FFT).

Stand-in statement: the paper trains on real LIGO O3 strain from GWOSC (PAPER.md:75, :93,
:103); that data is not available here, so stationary coloured Gaussian noise with the
analytic aLIGO fit stands in for it in every config.
"""
from dataclasses import dataclass, field

import numpy as np

PSD_SCALE_LOG2 = 140          # psd buffers of the C ABI hold S(f) * 2^140 (include/amplfi.h)
N_PARAMS = 11                 # mchirp q chi1 chi2 dist theta_jn phi_c t_c ra dec psi

H1, L1, V1 = 0, 1, 2


def aligo_psd(f):
    """BASELINE.json configs[0]: S(f) = 1e-49 [x^-4.14 - 5 x^-2 + 111 (1 - x^2 + x^4/2)/(1 + x^2/2)],
    x = f / 215 Hz, floored below 20 Hz (x = max(f, 20)/215)."""
    x = np.maximum(np.asarray(f, dtype=np.float64), 20.0) / 215.0
    return 1e-49 * (x ** -4.14 - 5.0 * x ** -2 + 111.0 * (1.0 - x * x + 0.5 * x ** 4) / (1.0 + 0.5 * x * x))


def coloured_noise(rng, shape, n, fs, dtype=np.float32):
    """Periodic stationary Gaussian noise with one-sided PSD aligo_psd: independent complex
    Gaussians with E|X_k|^2 = S(f_k) n fs / 2, real DC/Nyquist, inverse real FFT.  shape = leading dims."""
    k = n // 2 + 1
    f = np.arange(k) * (fs / n)
    sigma = np.sqrt(aligo_psd(f) * n * fs / 4.0)                # per real/imag component
    out = np.empty(tuple(shape) + (n,), dtype=dtype)
    flat = out.reshape(-1, n)
    for i in range(flat.shape[0]):
        re = rng.standard_normal(k)
        im = rng.standard_normal(k)
        xk = (re + 1j * im) * sigma
        xk[0] = re[0] * sigma[0] * np.sqrt(2.0)
        xk[-1] = re[-1] * sigma[-1] * np.sqrt(2.0)
        flat[i] = np.fft.irfft(xk, n).astype(dtype)
    return out


def draw_params(rng, batch, mc=(10.0, 100.0), q=(0.125, 1.0), dist=(100.0, 3000.0), dist_law="volume",
                spins=0.99, t_c=(5.5, 6.5)):
    """Table 1 priors: Mc uniform, q uniform, D_L ~ D^2 (or uniform), theta_JN sine,
    ra uniform, dec cosine, phi_c uniform(0, 2 pi), psi uniform(0, pi); aligned spins uniform in
    [-spins, spins] (BASELINE configs[1]); t_c uniform in the given window (time-shift up to 1 s,
    PAPER.md:93, :117)."""
    p = np.zeros((batch, N_PARAMS), dtype=np.float64)
    p[:, 0] = rng.uniform(mc[0], mc[1], batch)
    p[:, 1] = rng.uniform(q[0], q[1], batch)
    if spins > 0:
        p[:, 2] = rng.uniform(-spins, spins, batch)
        p[:, 3] = rng.uniform(-spins, spins, batch)
    u = rng.uniform(0.0, 1.0, batch)
    if dist_law == "volume":
        p[:, 4] = np.cbrt(dist[0] ** 3 + u * (dist[1] ** 3 - dist[0] ** 3))
    else:
        p[:, 4] = dist[0] + u * (dist[1] - dist[0])
    p[:, 5] = np.arccos(rng.uniform(-1.0, 1.0, batch))
    p[:, 6] = rng.uniform(0.0, 2.0 * np.pi, batch)
    p[:, 7] = rng.uniform(t_c[0], t_c[1], batch)
    p[:, 8] = rng.uniform(0.0, 2.0 * np.pi, batch)
    p[:, 9] = np.arcsin(rng.uniform(-1.0, 1.0, batch))
    p[:, 10] = rng.uniform(0.0, np.pi, batch)
    return p


@dataclass
class Workload:
    name: str
    batch: int
    det_ids: tuple
    fs: float
    n: int
    approximant: int              # 0 TaylorF2, 1 IMRPhenomD
    f_lo: float = 20.0
    f_hi: float = 1000.0
    gmst: float = 0.0
    nperseg: int = 0              # 0: PSD supplied on the segment grid
    params: np.ndarray = None     # [B, 11] fp64
    noise: np.ndarray = None      # dense [B, D, N] fp32, or None when gathered
    strip: np.ndarray = None      # [D, L] fp32
    offsets: np.ndarray = None    # [B, D] int64
    bg: np.ndarray = None         # [D, n_bg] fp32 background for Welch (None: analytic PSD)
    psd_scaled: np.ndarray = None # [D, K] fp32 = S * 2^140 (analytic-PSD configs)
    extra: dict = field(default_factory=dict)

    @property
    def n_det(self):
        return len(self.det_ids)


def _rng(seed):
    return np.random.Generator(np.random.Philox(seed))


def make_c0(batch=4, seed=0xA3D30000):
    """configs[0] "PR1 ref": batch 4, H1+L1, 2048 Hz, 4 s, TaylorF2 non-spinning, analytic PSD."""
    rng = _rng(seed)
    fs, n = 2048.0, 8192
    params = draw_params(rng, batch, mc=(10.0, 40.0), q=(0.25, 1.0), dist=(200.0, 1000.0),
                         dist_law="uniform", spins=0.0, t_c=(1.5, 2.5))
    noise = coloured_noise(rng, (batch, 2), n, fs)
    f = np.arange(n // 2 + 1) * (fs / n)
    psd = np.tile(aligo_psd(f) * 2.0 ** PSD_SCALE_LOG2, (2, 1)).astype(np.float32)
    return Workload("c0", batch, (H1, L1), fs, n, 0, params=params, noise=noise, psd_scaled=psd)


def make_c1(batch=256, seed=0xA3D30001, n=16384, fs=2048.0, bg_seconds=64, nperseg=4096):
    """configs[1]: batch 256, H1+L1+V1, 8 s, Welch from independent 64 s backgrounds, IMRPhenomD + spins."""
    rng = _rng(seed)
    t_seg = n / fs
    params = draw_params(rng, batch, t_c=(t_seg - 2.5, t_seg - 1.5))
    noise = coloured_noise(rng, (batch, 3), n, fs)
    bg = coloured_noise(rng, (3,), int(bg_seconds * fs), fs)
    return Workload("c1", batch, (H1, L1, V1), fs, n, 1, nperseg=nperseg, params=params, noise=noise, bg=bg)


def make_c2(batch=2048, seed=0xA3D30002, strip_len=44236800, n=16384, fs=2048.0, nperseg=4096,
            bg_seconds=64, align=1):
    """configs[2] training-throughput shape: noise gathered from a GPU-resident strip [3, L]
    (quarter day at 2048 Hz) at independent uniform offsets per (sample, detector);
    PSD per batch from a 64 s window of the strip at a random offset.  The strip is built by tiling
    a 2^22-sample periodic coloured-noise block (periodicity keeps it stationary across tiles)."""
    rng = _rng(seed)
    t_seg = n / fs
    params = draw_params(rng, batch, t_c=(t_seg - 2.5, t_seg - 1.5))
    block = 1 << 22
    base = coloured_noise(rng, (3,), min(block, strip_len), fs)
    reps = -(-strip_len // base.shape[-1])
    strip = np.tile(base, (1, reps))[:, :strip_len].copy()
    offsets = rng.integers(0, strip_len - n + 1, size=(batch, 3), dtype=np.int64)
    if align > 1:
        offsets -= offsets % align
    n_bg = int(bg_seconds * fs)
    bg_off = int(rng.integers(0, strip_len - n_bg + 1))
    return Workload("c2", batch, (H1, L1, V1), fs, n, 1, nperseg=nperseg, params=params, strip=strip,
                    offsets=offsets, extra={"bg_offset": bg_off, "n_bg": n_bg})


def make_c3(run=0, seed=0xA3D30003):
    """configs[3] online-latency shape: one candidate, 8 s segment + 128 s preceding background,
    nperseg 8192.  The distance rescaling to SNR 12 is done by the caller (it needs the method)."""
    rng = _rng(seed + run)
    fs, n, n_bg = 2048.0, 16384, 262144
    params = draw_params(rng, 1, t_c=(5.5, 6.5))
    data = coloured_noise(rng, (3,), n_bg + n, fs)               # background immediately precedes the segment
    bg = np.ascontiguousarray(data[:, :n_bg])
    noise = np.ascontiguousarray(data[:, n_bg:])[None]
    return Workload("c3", 1, (H1, L1, V1), fs, n, 1, nperseg=8192, params=params, noise=noise, bg=bg)


def make_c4(batch=8192, seed=0xA3D30004, t_seg=16.0, fs=4096.0, strip_len=1 << 26):
    """configs[4] bandwidth stress: fs 4096, 16 s (65536 samples), nperseg 16384 from 128 s background.
    Noise gathered from an 805 MB strip (offsets multiple of 4) so the full batch needs no 6.4 GB
    host array; sweep t_seg in {1,2,4,8,16} at fixed total samples by the caller."""
    rng = _rng(seed)
    n = int(t_seg * fs)
    params = draw_params(rng, batch, t_c=(max(t_seg - 2.5, 0.25 * t_seg), max(t_seg - 1.5, 0.5 * t_seg)))
    block = 1 << 22
    base = coloured_noise(rng, (3,), block, fs)
    strip = np.tile(base, (1, strip_len // block)).copy()
    offsets = rng.integers(0, strip_len - n + 1, size=(batch, 3), dtype=np.int64)
    offsets -= offsets % 4
    n_bg = int(128 * fs)
    return Workload("c4", batch, (H1, L1, V1), fs, n, 1, nperseg=16384, params=params, strip=strip,
                    offsets=offsets, extra={"bg_offset": 0, "n_bg": n_bg})
