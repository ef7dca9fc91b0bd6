"""Thin Python binding of libamplfi (include/amplfi.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of ``libamplfi.so``; torch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing, importing this
package raises, and every compute call needs CUDA tensors.

The functions keep the C names: ``amplfi_waveform_fd``, ``amplfi_project``, ``amplfi_psd_welch``,
``amplfi_inject_whiten`` (PAPER.md:101-105 for the steps they implement).
"""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libamplfi.so")

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED_SIZE, ERR_CUDA, ERR_ALIGNMENT = 0, -1, -2, -3, -4
TAYLORF2, IMRPHENOMD, SINE_GAUSSIAN = 0, 1, 2
H1, L1, V1 = 0, 1, 2
N_PARAMS = 11

EXPORTS = ("amplfi_last_error", "amplfi_psd_scale", "amplfi_version", "amplfi_phenomd_table",
           "amplfi_plan_create", "amplfi_plan_destroy", "amplfi_waveform_fd", "amplfi_project",
           "amplfi_psd_welch", "amplfi_inject_whiten", "amplfi_launch_count", "amplfi_plan_set_timing",
           "amplfi_plan_kernel_times", "amplfi_assemble_batch", "amplfi_probe_fp32_pipe",
           "amplfi_inject_whiten_views", "amplfi_waveform_td", "amplfi_inject_whiten_fir", "amplfi_qnm_table",
           "amplfi_psd_welch_noalloc")


class AmplfiError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libamplfi error %d: %s" % (code, msg))
        self.code = code


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError("libamplfi.so not found at %s: build it with `python paper_2407_19048_b200/build.py` "
                          "(there is no CPU fallback)" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    c = ctypes
    vp, dbl, i32, i64 = c.c_void_p, c.c_double, c.c_int, c.c_long
    lib.amplfi_last_error.restype = c.c_char_p
    lib.amplfi_last_error.argtypes = []
    lib.amplfi_psd_scale.restype = dbl
    lib.amplfi_psd_scale.argtypes = []
    lib.amplfi_version.restype = c.c_char_p
    lib.amplfi_version.argtypes = []
    lib.amplfi_launch_count.restype = i64
    lib.amplfi_launch_count.argtypes = []
    lib.amplfi_phenomd_table.restype = i32
    lib.amplfi_phenomd_table.argtypes = [vp]
    lib.amplfi_qnm_table.restype = i32
    lib.amplfi_qnm_table.argtypes = [vp]
    lib.amplfi_plan_create.restype = i32
    lib.amplfi_plan_create.argtypes = [i32, dbl, i32, c.POINTER(i32), i32, i32, c.POINTER(vp)]
    lib.amplfi_plan_destroy.restype = None
    lib.amplfi_plan_destroy.argtypes = [vp]
    lib.amplfi_plan_set_timing.restype = i32
    lib.amplfi_plan_set_timing.argtypes = [vp, i32]
    lib.amplfi_plan_kernel_times.restype = i32
    lib.amplfi_plan_kernel_times.argtypes = [vp, vp, i32]
    lib.amplfi_waveform_fd.restype = i32
    lib.amplfi_waveform_fd.argtypes = [vp, i32, i32, vp, dbl, dbl, vp, vp, vp, vp]
    lib.amplfi_project.restype = i32
    lib.amplfi_project.argtypes = [vp, i32, vp, dbl, vp, vp, vp, vp, vp]
    lib.amplfi_psd_welch.restype = i32
    lib.amplfi_psd_welch.argtypes = [vp, vp, i64, i64, i32, i32, i32, vp, vp]
    lib.amplfi_psd_welch_noalloc.restype = i32
    lib.amplfi_psd_welch_noalloc.argtypes = [vp, i64, i64, i32, dbl, i32, i32, i32, vp, vp]
    lib.amplfi_inject_whiten.restype = i32
    lib.amplfi_inject_whiten.argtypes = [vp, i32, vp, vp, i64, vp, i32, vp, dbl, vp, i32, dbl, dbl, vp, vp]
    lib.amplfi_probe_fp32_pipe.restype = i32
    lib.amplfi_probe_fp32_pipe.argtypes = [c.POINTER(dbl)]
    lib.amplfi_assemble_batch.restype = i32
    lib.amplfi_assemble_batch.argtypes = [vp, i32, vp, i64, i64, i32, i32, vp, vp, vp, i64, i32, vp, dbl, dbl, dbl, vp, vp]
    lib.amplfi_inject_whiten_views.restype = i32
    lib.amplfi_inject_whiten_views.argtypes = [vp, i32, vp, vp, i64, i32, vp, vp, dbl, vp, i32, dbl, dbl, vp, vp, vp]
    lib.amplfi_waveform_td.restype = i32
    lib.amplfi_waveform_td.argtypes = [vp, i32, i32, vp, dbl, dbl, vp, vp, vp]
    lib.amplfi_inject_whiten_fir.restype = i32
    lib.amplfi_inject_whiten_fir.argtypes = [vp, i32, vp, vp, i64, vp, i32, vp, dbl, vp, i32, dbl, dbl, dbl, i32, vp, vp]
    return lib


try:
    _lib = _load()
except AttributeError as exc:      # a symbol of include/amplfi.h is missing: the .so predates the sources
    raise ImportError("libamplfi.so is stale (%s): rebuild it with `python paper_2407_19048_b200/build.py --force`" % exc)


def _check(rc):
    if rc != OK:
        raise AmplfiError(rc, _lib.amplfi_last_error().decode())


def _ptr(t, dtype=None, name="tensor"):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA tensor (no CPU fallback)" % name)
    if dtype is not None and t.dtype != dtype:
        raise TypeError("%s must have dtype %s, got %s" % (name, dtype, t.dtype))
    if not t.is_contiguous():
        raise ValueError("%s must be contiguous" % name)
    return ctypes.c_void_p(t.data_ptr())


def _need(t, count, name):
    """The C ABI takes plain pointers: an undersized tensor would be an out-of-bounds device access, so sizes are checked here."""
    if t is not None and t.numel() < count:
        raise ValueError("%s holds %d elements, the call needs %d" % (name, t.numel(), count))


def _need_iw(plan, batch, noise, offsets, psd, h_det, params, out, n_out=None):
    nd, n, k = plan.n_det, plan.n, plan.n_bins
    if offsets is None:
        _need(noise, batch * nd * n, "noise")
    else:
        if noise.dim() != 2 or noise.shape[0] != nd:
            raise ValueError("with offsets, noise must be the strip [n_det, L]")
        _need(offsets, batch * nd, "offsets")
    if psd.dim() != 2 or psd.shape[0] != nd:
        raise ValueError("psd must be [n_det, n_psd]")
    _need(h_det, batch * nd * k * 2, "h_det")
    _need(params, batch * N_PARAMS, "params")
    _need(out, batch * nd * (n if n_out is None else n_out), "out")


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def last_error():
    return _lib.amplfi_last_error().decode()


def psd_scale():
    return _lib.amplfi_psd_scale()


def version():
    return _lib.amplfi_version().decode()


def launch_count():
    return int(_lib.amplfi_launch_count())


def phenomd_table():
    buf = (ctypes.c_double * 209)()
    _check(_lib.amplfi_phenomd_table(ctypes.cast(buf, ctypes.c_void_p)))
    return [list(buf[r * 11:(r + 1) * 11]) for r in range(19)]


def qnm_table():
    """(spins, Re M omega, -Im M omega) of the Kerr (2,2,0) mode as the library tabulates it (host computation, no GPU)."""
    buf = (ctypes.c_double * 1024)()
    n = _lib.amplfi_qnm_table(ctypes.cast(buf, ctypes.c_void_p))
    if n < 0:
        _check(n)
    y_lo, y_hi = (1.0 - 0.998) ** 0.5, (1.0 + 0.998) ** 0.5
    spins = [1.0 - (y_lo + (y_hi - y_lo) * i / (n - 1)) ** 2 for i in range(n)]
    return spins, [buf[2 * i] for i in range(n)], [buf[2 * i + 1] for i in range(n)]


class Plan:
    """amplfi_plan_create / amplfi_plan_destroy."""

    def __init__(self, n, fs, det_ids, max_batch, nperseg=0):
        det_ids = [int(d) for d in det_ids]
        arr = (ctypes.c_int * max(len(det_ids), 1))(*det_ids)
        handle = ctypes.c_void_p()
        _check(_lib.amplfi_plan_create(int(n), float(fs), len(det_ids), arr, int(max_batch), int(nperseg),
                                       ctypes.byref(handle)))
        self._h = handle
        self.n, self.fs, self.det_ids, self.max_batch, self.nperseg = int(n), float(fs), det_ids, int(max_batch), int(nperseg)
        self.n_det = len(det_ids)
        self.n_bins = self.n // 2 + 1

    def set_timing(self, enable=True):
        _check(_lib.amplfi_plan_set_timing(self._h, 1 if enable else 0))

    def kernel_times_ms(self, max_count=512):
        """Durations (ms) of the fused inject+whiten kernel of the calls made since set_timing(True)."""
        buf = (ctypes.c_float * max_count)()
        n = _lib.amplfi_plan_kernel_times(self._h, ctypes.cast(buf, ctypes.c_void_p), max_count)
        if n < 0:
            _check(n)
        return [float(buf[i]) for i in range(n)]

    def close(self):
        if getattr(self, "_h", None):
            _lib.amplfi_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def amplfi_waveform_fd(plan, approximant, params, f_lo, f_hi, hp=None, hc=None, flags=None, stream=None):
    """params [B, 11] fp64 cuda -> (hp, hc) [B, K, 2] fp32, flags [B] int32."""
    batch = params.shape[0]
    dev = params.device
    if hp is None:
        hp = torch.empty((batch, plan.n_bins, 2), dtype=torch.float32, device=dev)
    if hc is None:
        hc = torch.empty((batch, plan.n_bins, 2), dtype=torch.float32, device=dev)
    if flags is None:
        flags = torch.empty((batch,), dtype=torch.int32, device=dev)
    _need(params, batch * N_PARAMS, "params"); _need(hp, batch * plan.n_bins * 2, "hp"); _need(hc, batch * plan.n_bins * 2, "hc")
    _need(flags, batch, "flags")
    _check(_lib.amplfi_waveform_fd(plan._h, int(approximant), int(batch), _ptr(params, torch.float64, "params"),
                                   float(f_lo), float(f_hi), _ptr(hp, torch.float32, "hp"),
                                   _ptr(hc, torch.float32, "hc"), _ptr(flags, torch.int32, "flags"), _stream(stream)))
    return hp, hc, flags


def amplfi_project(plan, params, gmst, hp=None, hc=None, h_det=None, resp=None, want_resp=True, stream=None):
    """-> (h_det [B, D, K, 2] fp32 or None, resp [B, D, 3] fp64 or None)."""
    batch = params.shape[0]
    dev = params.device
    if hp is not None and h_det is None:
        h_det = torch.empty((batch, plan.n_det, plan.n_bins, 2), dtype=torch.float32, device=dev)
    if want_resp and resp is None:
        resp = torch.empty((batch, plan.n_det, 3), dtype=torch.float64, device=dev)
    _need(params, batch * N_PARAMS, "params"); _need(hp, batch * plan.n_bins * 2, "hp"); _need(hc, batch * plan.n_bins * 2, "hc")
    _need(h_det, batch * plan.n_det * plan.n_bins * 2, "h_det"); _need(resp, batch * plan.n_det * 3, "resp")
    _check(_lib.amplfi_project(plan._h, int(batch), _ptr(params, torch.float64, "params"), float(gmst),
                               _ptr(hp, torch.float32, "hp"), _ptr(hc, torch.float32, "hc"),
                               _ptr(h_det, torch.float32, "h_det"), _ptr(resp, torch.float64, "resp"),
                               _stream(stream)))
    return h_det, resp


def amplfi_psd_welch(plan, bg, noverlap=None, detrend=1, average=0, psd=None, stream=None):
    """bg [D, n_bg] fp32 -> psd [D, nperseg/2+1] fp32 (S * 2^140)."""
    if noverlap is None:
        noverlap = plan.nperseg // 2
    if psd is None:
        psd = torch.empty((plan.n_det, plan.nperseg // 2 + 1), dtype=torch.float32, device=bg.device)
    if bg.dim() != 2 or bg.shape[0] != plan.n_det or bg.stride(1) != 1:
        raise ValueError("bg must be [n_det, n_bg] with unit stride along time (rows may be a window of a strip)")
    if not bg.is_cuda or bg.dtype != torch.float32:
        raise TypeError("bg must be a CUDA float32 tensor (no CPU fallback)")
    row_stride = int(bg.stride(0)) if plan.n_det > 1 else int(bg.shape[1])
    _need(psd, plan.n_det * (plan.nperseg // 2 + 1), "psd")
    _check(_lib.amplfi_psd_welch(plan._h, ctypes.c_void_p(bg.data_ptr()), int(bg.shape[1]), row_stride, int(noverlap), int(detrend),
                                 int(average), _ptr(psd, torch.float32, "psd"), _stream(stream)))
    return psd


NOALLOC_WELCH_FLOATS = 1 << 20


def amplfi_psd_welch_noalloc(bg, fs, nperseg, psd, noverlap=None, detrend=1, stream=None):
    """bg [D, n_bg] fp32 -> psd [D, nperseg/2+1] fp32 (S * 2^140), caller-supplied: no plan, no device allocation (the
    library's static scratch array; see include/amplfi.h for its limit and the rule about overlapping calls)."""
    if noverlap is None:
        noverlap = nperseg // 2
    if bg.dim() != 2 or bg.stride(1) != 1:
        raise ValueError("bg must be [n_det, n_bg] with unit stride along time (rows may be a window of a strip)")
    if not bg.is_cuda or bg.dtype != torch.float32:
        raise TypeError("bg must be a CUDA float32 tensor (no CPU fallback)")
    n_det = int(bg.shape[0])
    row_stride = int(bg.stride(0)) if n_det > 1 else int(bg.shape[1])
    _need(psd, n_det * (nperseg // 2 + 1), "psd")
    _check(_lib.amplfi_psd_welch_noalloc(ctypes.c_void_p(bg.data_ptr()), int(bg.shape[1]), row_stride, n_det, float(fs),
                                         int(nperseg), int(noverlap), int(detrend), _ptr(psd, torch.float32, "psd"),
                                         _stream(stream)))
    return psd


def amplfi_inject_whiten(plan, batch, noise, psd, f_lo, f_hi, offsets=None, h_det=None, approximant=IMRPHENOMD,
                         params=None, gmst=0.0, out=None, stream=None):
    """noise dense [B, D, N] (offsets None) or strip [D, L] with offsets [B, D] int64 -> out [B, D, N] fp32."""
    if out is None:
        out = torch.empty((batch, plan.n_det, plan.n), dtype=torch.float32, device=noise.device)
    strip_len = int(noise.shape[-1]) if offsets is not None else 0
    _need_iw(plan, batch, noise, offsets, psd, h_det, params, out)
    _check(_lib.amplfi_inject_whiten(plan._h, int(batch), _ptr(noise, torch.float32, "noise"),
                                     _ptr(offsets, torch.int64, "offsets"), strip_len,
                                     _ptr(h_det, torch.float32, "h_det"), int(approximant),
                                     _ptr(params, torch.float64, "params"), float(gmst),
                                     _ptr(psd, torch.float32, "psd"), int(psd.shape[-1]), float(f_lo), float(f_hi),
                                     _ptr(out, torch.float32, "out"), _stream(stream)))
    return out


def amplfi_inject_whiten_views(plan, batch, noise, psd, f_lo, f_hi, params, t_shift, offsets=None, approximant=IMRPHENOMD,
                               gmst=0.0, out=None, out2=None, stream=None):
    """Two views (d, d') of PAPER.md:93, :117: out2 repeats out with t_c + t_shift[b].  -> (out, out2) [B, D, N] fp32."""
    if out is None:
        out = torch.empty((batch, plan.n_det, plan.n), dtype=torch.float32, device=noise.device)
    if out2 is None:
        out2 = torch.empty((batch, plan.n_det, plan.n), dtype=torch.float32, device=noise.device)
    strip_len = int(noise.shape[-1]) if offsets is not None else 0
    _need_iw(plan, batch, noise, offsets, psd, None, params, out)
    _need(out2, batch * plan.n_det * plan.n, "out2"); _need(t_shift, batch, "t_shift")
    _check(_lib.amplfi_inject_whiten_views(plan._h, int(batch), _ptr(noise, torch.float32, "noise"),
                                           _ptr(offsets, torch.int64, "offsets"), strip_len, int(approximant),
                                           _ptr(params, torch.float64, "params"), _ptr(t_shift, torch.float64, "t_shift"),
                                           float(gmst), _ptr(psd, torch.float32, "psd"), int(psd.shape[-1]), float(f_lo),
                                           float(f_hi), _ptr(out, torch.float32, "out"), _ptr(out2, torch.float32, "out2"),
                                           _stream(stream)))
    return out, out2


def amplfi_waveform_td(plan, approximant, params, f_lo, f_hi, h_t=None, flags=None, stream=None):
    """params [B, 11] fp64 cuda -> h_t [B, 2, N] fp32 (row 0 h+(t), row 1 hx(t)), flags [B] int32."""
    batch = params.shape[0]
    if h_t is None:
        h_t = torch.empty((batch, 2, plan.n), dtype=torch.float32, device=params.device)
    if flags is None:
        flags = torch.empty((batch,), dtype=torch.int32, device=params.device)
    _need(params, batch * N_PARAMS, "params"); _need(h_t, batch * 2 * plan.n, "h_t"); _need(flags, batch, "flags")
    _check(_lib.amplfi_waveform_td(plan._h, int(approximant), int(batch), _ptr(params, torch.float64, "params"), float(f_lo),
                                   float(f_hi), _ptr(h_t, torch.float32, "h_t"), _ptr(flags, torch.int32, "flags"),
                                   _stream(stream)))
    return h_t, flags


def amplfi_inject_whiten_fir(plan, batch, noise, psd, f_lo, f_hi, fduration, crop=True, offsets=None, h_det=None,
                             approximant=IMRPHENOMD, params=None, gmst=0.0, out=None, stream=None):
    """amplfi_inject_whiten with the whitening filter truncated to fduration seconds; crop drops fduration/2 at each
    end -> out [B, D, N - fduration*fs] (crop) or [B, D, N]."""
    ntaps = int(round(fduration * plan.fs))
    n_out = max(plan.n - ntaps, 2) if crop else plan.n      # invalid fduration: the library reports it
    if out is None:
        out = torch.empty((batch, plan.n_det, n_out), dtype=torch.float32, device=noise.device)
    strip_len = int(noise.shape[-1]) if offsets is not None else 0
    _need_iw(plan, batch, noise, offsets, psd, h_det, params, out, n_out)
    _check(_lib.amplfi_inject_whiten_fir(plan._h, int(batch), _ptr(noise, torch.float32, "noise"),
                                         _ptr(offsets, torch.int64, "offsets"), strip_len,
                                         _ptr(h_det, torch.float32, "h_det"), int(approximant),
                                         _ptr(params, torch.float64, "params"), float(gmst),
                                         _ptr(psd, torch.float32, "psd"), int(psd.shape[-1]), float(f_lo), float(f_hi),
                                         float(fduration), 1 if crop else 0, _ptr(out, torch.float32, "out"),
                                         _stream(stream)))
    return out


def amplfi_assemble_batch(plan, batch, bg, noise, params, f_lo, f_hi, offsets=None, approximant=IMRPHENOMD, gmst=0.0,
                          noverlap=None, detrend=1, psd=None, out=None, stream=None):
    """One data-generation step: Welch PSD of bg [D, n_bg], then waveform generation, projection, injection into
    noise (dense [B, D, N], or strip [D, L] with offsets [B, D]) and whitening -> (out [B, D, N], psd)."""
    if noverlap is None:
        noverlap = plan.nperseg // 2
    if psd is None:
        psd = torch.empty((plan.n_det, plan.nperseg // 2 + 1), dtype=torch.float32, device=bg.device)
    if out is None:
        out = torch.empty((batch, plan.n_det, plan.n), dtype=torch.float32, device=noise.device)
    if bg.dim() != 2 or bg.shape[0] != plan.n_det or bg.stride(1) != 1:
        raise ValueError("bg must be [n_det, n_bg] with unit stride along time (rows may be a window of a strip)")
    if not bg.is_cuda or bg.dtype != torch.float32:
        raise TypeError("bg must be a CUDA float32 tensor (no CPU fallback)")
    row_stride = int(bg.stride(0)) if plan.n_det > 1 else int(bg.shape[1])
    strip_len = int(noise.shape[-1]) if offsets is not None else 0
    _need_iw(plan, batch, noise, offsets, psd, None, params, out)
    _check(_lib.amplfi_assemble_batch(plan._h, int(batch), ctypes.c_void_p(bg.data_ptr()), int(bg.shape[1]), row_stride,
                                      int(noverlap), int(detrend), _ptr(psd, torch.float32, "psd"),
                                      _ptr(noise, torch.float32, "noise"), _ptr(offsets, torch.int64, "offsets"),
                                      strip_len, int(approximant), _ptr(params, torch.float64, "params"), float(gmst),
                                      float(f_lo), float(f_hi), _ptr(out, torch.float32, "out"), _stream(stream)))
    return out, psd


def probe_fp32_pipe():
    """Measured fp32 lane-operations per second of the current device (packed FMA loop on every SM)."""
    v = ctypes.c_double(0.0)
    _check(_lib.amplfi_probe_fp32_pipe(ctypes.byref(v)))
    return float(v.value)
