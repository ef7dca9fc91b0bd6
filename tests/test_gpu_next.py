"""GPU parity of the SURVEY.md 8(f) calls against the oracle: two data views, time-domain waveform
output, median-averaged Welch and the time-truncated whitening filter.  Same tolerances as
tests/test_gpu_parity.py (BASELINE.json north_star): 1e-4 of the row RMS on strain, 1e-4 relative on the PSD in band."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

if not torch.cuda.is_available():
    pytest.skip("needs a CUDA device", allow_module_level=True)

import paper_2407_19048_b200 as A          # noqa: E402
import workloads as WL                     # noqa: E402
from oracle import project as OP           # noqa: E402
from oracle import views as OV             # noqa: E402
from oracle import waveform as OW          # noqa: E402
from oracle import welch as OWE            # noqa: E402
from oracle import whiten as OWH           # noqa: E402

from test_gpu_parity import TOL, PSD_SCALE, dev, row_err, edge_params      # noqa: E402


def _make_inputs(n, fs, batch, dets, seed):
    rng = np.random.Generator(np.random.Philox(seed))
    t_seg = n / fs
    par = WL.draw_params(rng, batch, t_c=(t_seg - 2.5, t_seg - 1.5) if t_seg >= 4 else (0.5 * t_seg, 0.6 * t_seg))
    noise = WL.coloured_noise(rng, (batch, len(dets)), n, fs)
    psd = np.stack([WL.aligo_psd(np.arange(n // 2 + 1) * fs / n) * (1.0 + 0.1 * d) for d in range(len(dets))])
    return par, noise, psd


# ------------------------------------------------------------------------------------------ two views
@pytest.mark.parametrize("n,fs,approx", [(16384, 2048.0, A.IMRPHENOMD), (8192, 2048.0, A.TAYLORF2), (65536, 4096.0, A.IMRPHENOMD),
                                         (2048, 2048.0, A.IMRPHENOMD), (4096, 2048.0, A.IMRPHENOMD), (8192, 4096.0, A.IMRPHENOMD),
                                         (131072, 4096.0, A.IMRPHENOMD), (262144, 4096.0, A.IMRPHENOMD)])
def test_two_views_parity(n, fs, approx):
    dets = [0, 1, 2]
    batch = 6
    par, noise, psd = _make_inputs(n, fs, batch, dets, 1000 + n)
    par[0, 4] = 100.0                                         # one very loud signal: phase errors would show
    t_shift = np.array([1.0, 0.0, 0.37, 1.0 / fs, 0.999, 0.5])[:batch]
    plan = A.Plan(n, fs, dets, batch)
    out, out2 = A.amplfi_inject_whiten_views(plan, batch, dev(noise), dev((psd * PSD_SCALE).astype(np.float32)), 20.0, 1000.0,
                                             dev(par), dev(t_shift), approximant=approx, gmst=0.3)
    torch.cuda.synchronize()
    psd32 = (psd * PSD_SCALE).astype(np.float32).astype(np.float64) / PSD_SCALE
    d, d2 = OV.two_views(approx, par, t_shift, noise.astype(np.float64), psd32, 0.3, dets, fs, 20.0, 1000.0)
    assert row_err(out.cpu().numpy().astype(np.float64), d).max() <= TOL
    assert row_err(out2.cpu().numpy().astype(np.float64), d2).max() <= TOL
    # the signal part alone (noise removed on both sides) to the same bar relative to ITS rms
    bg = A.amplfi_inject_whiten(plan, batch, dev(noise), dev((psd * PSD_SCALE).astype(np.float32)), 20.0, 1000.0)
    bg_ref = OWH.inject_whiten(noise.astype(np.float64), None, psd32, fs, 20.0, 1000.0)
    s_gpu = (out2 - bg).cpu().numpy().astype(np.float64)
    s_ref = d2 - bg_ref
    assert row_err(s_gpu[0], s_ref[0]).max() <= 2e-3           # difference of two fp32 rows: noise rounding remains
    # zero shift reproduces the first view bit for bit
    assert torch.equal(out[1], out2[1])


def test_two_views_from_strip_with_offsets():
    wl = WL.make_c2(batch=8, strip_len=1 << 20)
    plan = A.Plan(wl.n, wl.fs, wl.det_ids, 8, nperseg=wl.nperseg)
    o, nb = wl.extra["bg_offset"], wl.extra["n_bg"]
    psd = A.amplfi_psd_welch(plan, dev(np.ascontiguousarray(wl.strip[:, o:o + nb])))
    t_shift = np.linspace(0.0, 1.0, 8)
    out, out2 = A.amplfi_inject_whiten_views(plan, 8, dev(wl.strip), psd, wl.f_lo, wl.f_hi, dev(wl.params[:8]), dev(t_shift),
                                             offsets=dev(wl.offsets[:8]), gmst=wl.gmst)
    torch.cuda.synchronize()
    psd_ref = psd.cpu().numpy().astype(np.float64) / PSD_SCALE
    noise = OWH.gather(wl.strip, wl.offsets[:8], wl.n)
    d, d2 = OV.two_views(wl.approximant, wl.params[:8], t_shift, noise, psd_ref, wl.gmst, wl.det_ids, wl.fs, wl.f_lo, wl.f_hi)
    assert row_err(out.cpu().numpy().astype(np.float64), d).max() <= TOL
    assert row_err(out2.cpu().numpy().astype(np.float64), d2).max() <= TOL


@pytest.mark.parametrize("n", [4096, 8192, 16384, 2048])
def test_two_views_out_of_range_offset_poisons_both_views(n):
    """include/amplfi.h: an out-of-range gather offset gives an all-NaN row -- in BOTH views (the one-launch two-view
    kernel of n = 4096 .. 16384 and the two-launch path of the other lengths), every other row finite."""
    fs = 2048.0
    dets = [0, 1, 2]
    batch = 4
    par, _, psd = _make_inputs(n, fs, batch, dets, 7000 + n)
    rng = np.random.Generator(np.random.Philox(n + 11))
    strip = WL.coloured_noise(rng, (3,), 1 << 18, fs)
    offsets = rng.integers(0, strip.shape[1] - n, size=(batch, 3)).astype(np.int64)
    offsets[1, 0] = strip.shape[1] - n + 1
    offsets[2, 2] = -1
    plan = A.Plan(n, fs, dets, batch)
    out, out2 = A.amplfi_inject_whiten_views(plan, batch, dev(strip), dev((psd * PSD_SCALE).astype(np.float32)), 20.0, 1000.0,
                                             dev(par), dev(np.full(batch, 0.25)), offsets=dev(offsets))
    torch.cuda.synchronize()
    bad = np.zeros((batch, 3), bool)
    bad[1, 0] = bad[2, 2] = True
    for o in (out, out2):
        g = o.cpu().numpy()
        assert np.all(np.isnan(g[bad])) and np.all(np.isfinite(g[~bad]))


# ------------------------------------------------------------------------------------------ time-domain waveform
@pytest.mark.parametrize("approx", [A.TAYLORF2, A.IMRPHENOMD])
@pytest.mark.parametrize("n,fs", [(8192, 2048.0), (16384, 2048.0), (65536, 4096.0), (1024, 2048.0), (4096, 2048.0), (131072, 4096.0),
                                   (262144, 4096.0)])
def test_waveform_td_parity(approx, n, fs):
    par = edge_params(0.6 * n / fs)
    par = np.concatenate([par, par[:1]])
    par[-1, 1] = 1.5                                          # invalid q: all-zero row and a flag
    plan = A.Plan(n, fs, [0], len(par))
    h_t, flags = A.amplfi_waveform_td(plan, approx, dev(par), 20.0, 1000.0)
    torch.cuda.synchronize()
    hp, hc, fl = OW.waveform_td(approx, par, n, fs, 20.0, 1000.0)
    got = h_t.cpu().numpy().astype(np.float64)
    assert np.array_equal(flags.cpu().numpy(), fl)
    assert row_err(got[:, 0], hp).max() <= TOL
    assert row_err(got[:, 1], hc).max() <= TOL
    assert np.all(got[-1] == 0.0)


# ------------------------------------------------------------------------------------------ median Welch
@pytest.mark.parametrize("nperseg,n_bg,fs", [(4096, 131072, 2048.0), (8192, 262144, 2048.0), (1024, 1024 * 32 + 512, 2048.0),
                                             (1024, 1024, 2048.0), (2048, 2048 * 128 + 1024, 4096.0)])
def test_welch_median_parity(nperseg, n_bg, fs):
    rng = np.random.Generator(np.random.Philox(nperseg + 7))
    bg = WL.coloured_noise(rng, (3,), 1 << 19, fs)[:, :n_bg].copy()
    bg[1, 5000:5040] += np.float32(4e-19)                      # a loud transient the median should ignore
    plan = A.Plan(max(nperseg, 1024), fs, [0, 1, 2], 1, nperseg=nperseg)
    psd = A.amplfi_psd_welch(plan, dev(bg), average=1)
    assert torch.equal(psd, A.amplfi_psd_welch(plan, dev(bg), average=1))
    ref = OWE.welch(bg.astype(np.float64), fs, nperseg, average="median") * PSD_SCALE
    got = psd.cpu().numpy().astype(np.float64)
    f = np.arange(nperseg // 2 + 1) * fs / nperseg
    band = (f >= 20.0) & (f <= 1000.0)
    level = WL.aligo_psd(f) * PSD_SCALE
    assert (np.abs(got - ref)[:, band] / level[band]).max() <= TOL
    nseg = (n_bg - nperseg) // (nperseg // 2) + 1
    if nseg >= 8:
        assert np.abs(got[:, band] / ref[:, band] - 1).max() <= TOL


# ------------------------------------------------------------------------------------------ truncated whitening filter
@pytest.mark.parametrize("n,fs,fdur", [(16384, 2048.0, 1.0), (8192, 2048.0, 0.5), (65536, 4096.0, 2.0), (2048, 2048.0, 0.25),
                                       (16384, 2048.0, 8.0), (4096, 2048.0, 0.5), (131072, 4096.0, 2.0),
                                       (262144, 4096.0, 2.0)])
@pytest.mark.parametrize("crop", [True, False])
def test_inject_whiten_fir_parity(n, fs, fdur, crop):
    if crop and fdur * fs >= n:
        pytest.skip("nothing left after cropping")
    dets = [0, 1]
    batch = 3
    par, noise, psd = _make_inputs(n, fs, batch, dets, 2000 + n)
    psd = psd * (1.0 + 0.5 * np.sin(np.arange(n // 2 + 1) / 7.0) ** 2)      # a structured PSD: truncation matters
    psd_s = (psd * PSD_SCALE).astype(np.float32)
    plan = A.Plan(n, fs, dets, batch)
    out = A.amplfi_inject_whiten_fir(plan, batch, dev(noise), dev(psd_s), 20.0, 1000.0, fdur, crop=crop, params=dev(par), gmst=0.1)
    torch.cuda.synchronize()
    psd64 = psd_s.astype(np.float64) / PSD_SCALE
    hp, hc, _ = OW.waveform_fd(A.IMRPHENOMD, par, n, fs, 20.0, 1000.0)
    h_det, _ = OP.project(hp, hc, par, 0.1, dets, n, fs)
    ref = OWH.inject_whiten_fir(noise.astype(np.float64), h_det, psd64, fs, 20.0, 1000.0, fdur, crop=crop)
    got = out.cpu().numpy().astype(np.float64)
    assert got.shape == ref.shape
    assert row_err(got, ref).max() <= TOL
    # whiten only, h_det given: the other two modes of the call
    out_n = A.amplfi_inject_whiten_fir(plan, batch, dev(noise), dev(psd_s), 20.0, 1000.0, fdur, crop=crop)
    ref_n = OWH.inject_whiten_fir(noise.astype(np.float64), None, psd64, fs, 20.0, 1000.0, fdur, crop=crop)
    assert row_err(out_n.cpu().numpy().astype(np.float64), ref_n).max() <= TOL


def test_fir_argument_checks():
    plan = A.Plan(4096, 2048.0, [0], 1)
    noise = torch.zeros((1, 1, 4096), device="cuda")
    psd = torch.ones((1, 2049), device="cuda")
    for fdur in (0.0, 3.0, 0.5 + 1.0 / 2048.0):
        with pytest.raises(A.AmplfiError):
            A.amplfi_inject_whiten_fir(plan, 1, noise, psd, 20.0, 1000.0, fdur)
    with pytest.raises(A.AmplfiError):
        A.amplfi_inject_whiten_fir(plan, 1, noise, psd, 20.0, 1000.0, 2.0, crop=True)


# ------------------------------------------------------------------------------------------ degenerate rows of the fused path
@pytest.mark.parametrize("n,fs", [(16384, 2048.0), (8192, 2048.0), (65536, 4096.0)])
def test_fused_invalid_and_empty_band_rows_inject_nothing(n, fs):
    """A sample with invalid parameters, or whose band is empty (f_top < f_lo: reading R-W7), must come out exactly as
    whitened noise, even when the plan's h0 workspace still holds a previous, loud batch."""
    dets = [0, 1, 2]
    batch = 4
    par, noise, psd = _make_inputs(n, fs, batch, dets, 3000 + n)
    par[:, 4] = 50.0                                           # loud batch that fills the workspace
    psd_s = dev((psd * PSD_SCALE).astype(np.float32))
    plan = A.Plan(n, fs, dets, batch)
    A.amplfi_inject_whiten(plan, batch, dev(noise), psd_s, 20.0, 1000.0, params=dev(par))
    bad = par.copy()
    bad[0, 1] = 1.5                                            # q > 1
    bad[1, 2] = 1.0                                            # |chi1| = 1
    bad[2, 0], bad[2, 1] = 100.0, 1.0                          # TaylorF2: f_ISCO = 19.1 Hz < f_lo -> empty band
    bad[3, 4] = -1.0                                           # distance <= 0
    out = A.amplfi_inject_whiten(plan, batch, dev(noise), psd_s, 20.0, 1000.0, approximant=A.TAYLORF2, params=dev(bad))
    ref = A.amplfi_inject_whiten(plan, batch, dev(noise), psd_s, 20.0, 1000.0)
    torch.cuda.synchronize()
    assert torch.equal(out, ref)


# ------------------------------------------------------------------------------------------ long segments (8(f)-4)
@pytest.mark.parametrize("n,fs,mode", [(1 << 17, 4096.0, "fused"), (1 << 17, 4096.0, "none"), (1 << 18, 4096.0, "fused"),
                                       (1 << 18, 4096.0, "hdet"), (1 << 19, 4096.0, "fused"), (1 << 20, 4096.0, "fused")])
def test_long_segments_parity(n, fs, mode):
    """binary-neutron-star signals last minutes, "input arrays larger by an order of magnitude": segments of
    32 .. 256 s at 4096 Hz, a low-mass TaylorF2 inspiral that spends the whole segment in band next to a heavy IMR system."""
    dets = [0, 1]
    batch = 2
    t_seg = n / fs
    rng = np.random.Generator(np.random.Philox(n))
    par = WL.draw_params(rng, batch, t_c=(t_seg - 2.5, t_seg - 1.5))
    par[0, :5] = [1.2, 0.9, 0.0, 0.0, 40.0]                    # a binary neutron star at 40 Mpc
    approx = A.TAYLORF2
    noise = WL.coloured_noise(rng, (batch, len(dets)), n, fs)
    psd = np.stack([WL.aligo_psd(np.arange(n // 2 + 1) * fs / n)] * 2)
    psd_s = (psd * PSD_SCALE).astype(np.float32)
    plan = A.Plan(n, fs, dets, batch)
    kw = {}
    h_det_ref = None
    if mode != "none":
        hp, hc, _ = OW.waveform_fd(approx, par, n, fs, 20.0, 1000.0)
        h_det_ref, _ = OP.project(hp, hc, par, 0.2, dets, n, fs)
    if mode == "fused":
        kw = dict(approximant=approx, params=dev(par), gmst=0.2)
    elif mode == "hdet":
        hp_g, hc_g, _ = A.amplfi_waveform_fd(plan, approx, dev(par), 20.0, 1000.0)
        h_det, _ = A.amplfi_project(plan, dev(par), 0.2, hp_g, hc_g)
        kw = dict(h_det=h_det)
    out = A.amplfi_inject_whiten(plan, batch, dev(noise), dev(psd_s), 20.0, 1000.0, **kw)
    torch.cuda.synchronize()
    ref = OWH.inject_whiten(noise.astype(np.float64), h_det_ref, psd_s.astype(np.float64) / PSD_SCALE, fs, 20.0, 1000.0)
    assert row_err(out.cpu().numpy().astype(np.float64), ref).max() <= TOL


def test_long_segment_gather_views_and_td():
    """n = 2^17 through the other entry points: strip gather with offsets, two views, time-domain output, cropped FIR."""
    n, fs, dets, batch = 1 << 17, 4096.0, [0, 1, 2], 2
    rng = np.random.Generator(np.random.Philox(17))
    par = WL.draw_params(rng, batch, t_c=(29.0, 30.0))
    strip = WL.coloured_noise(rng, (3,), 1 << 19, fs)
    offsets = np.array([[5, 100001, 262144 + 3], [393216, 0, 77]], dtype=np.int64)
    psd = np.stack([WL.aligo_psd(np.arange(n // 2 + 1) * fs / n)] * 3)
    psd_s = (psd * PSD_SCALE).astype(np.float32)
    psd64 = psd_s.astype(np.float64) / PSD_SCALE
    plan = A.Plan(n, fs, dets, batch)
    t_shift = np.array([0.75, 0.001])
    out, out2 = A.amplfi_inject_whiten_views(plan, batch, dev(strip), dev(psd_s), 20.0, 1000.0, dev(par), dev(t_shift),
                                             offsets=dev(offsets), gmst=0.4)
    noise = OWH.gather(strip, offsets, n)
    d, d2 = OV.two_views(A.IMRPHENOMD, par, t_shift, noise, psd64, 0.4, dets, fs, 20.0, 1000.0)
    assert row_err(out.cpu().numpy().astype(np.float64), d).max() <= TOL
    assert row_err(out2.cpu().numpy().astype(np.float64), d2).max() <= TOL
    h_t, _ = A.amplfi_waveform_td(plan, A.IMRPHENOMD, dev(par), 20.0, 1000.0)
    hp, hc, _ = OW.waveform_td(A.IMRPHENOMD, par, n, fs, 20.0, 1000.0)
    got = h_t.cpu().numpy().astype(np.float64)
    assert row_err(got[:, 0], hp).max() <= TOL and row_err(got[:, 1], hc).max() <= TOL
    out_f = A.amplfi_inject_whiten_fir(plan, batch, dev(strip), dev(psd_s), 20.0, 1000.0, 2.0, crop=True, offsets=dev(offsets))
    ref_f = OWH.inject_whiten_fir(noise, None, psd64, fs, 20.0, 1000.0, 2.0, crop=True)
    assert row_err(out_f.cpu().numpy().astype(np.float64), ref_f).max() <= TOL


# ------------------------------------------------------------------------------------------ sine-Gaussian family (8(f)-4)
def _sg_params(n, fs):
    t_seg = n / fs
    rows = []
    for f0, q, amp, iota in [(250.0, 9.0, 1e-21, 0.6), (60.0, 4.0, 5e-22, 0.0), (800.0, 100.0, 2e-21, 1.5707963),
                             (35.0, 20.0, 1e-20, 2.5), (999.0, 3.0, 1e-21, 1.0), (250.0, -1.0, 1e-21, 0.3)]:
        rows.append([f0, q, 0.0, 0.0, amp, iota, 1.3, 0.55 * t_seg, 1.0, 0.5, 0.7])
    return np.array(rows, dtype=np.float64)


@pytest.mark.parametrize("n,fs", [(16384, 2048.0), (8192, 2048.0), (65536, 4096.0)])
def test_sine_gaussian_parity(n, fs):
    par = _sg_params(n, fs)
    dets = [0, 1, 2]
    plan = A.Plan(n, fs, dets, len(par))
    hp, hc, flags = A.amplfi_waveform_fd(plan, A.SINE_GAUSSIAN, dev(par), 20.0, 1000.0)
    hp_r, hc_r, fl_r = OW.waveform_fd(OW.SINE_GAUSSIAN, par, n, fs, 20.0, 1000.0)
    assert np.array_equal(flags.cpu().numpy(), fl_r)
    from test_gpu_parity import cplx
    assert row_err(cplx(hp), hp_r).max() <= TOL and row_err(cplx(hc), hc_r).max() <= TOL
    f = np.arange(n // 2 + 1) * fs / n
    outside = (f < 20.0) | (f > 1000.0)
    assert np.all(cplx(hp)[:, outside] == 0) and np.all(cplx(hc)[:, outside] == 0)      # hard band edges (R-W7)
    assert np.all(cplx(hp)[-1] == 0) and np.all(cplx(hc)[-1] == 0)                      # the invalid row
    assert cplx(hp)[4][f == 1000.0] != 0                                                # upper edge inclusive (f0 = 999 Hz)
    # injected and whitened through the fused call, and as a time series
    rng = np.random.Generator(np.random.Philox(n + 5))
    noise = WL.coloured_noise(rng, (len(par), 3), n, fs)
    psd = np.stack([WL.aligo_psd(np.arange(n // 2 + 1) * fs / n)] * 3)
    psd_s = (psd * PSD_SCALE).astype(np.float32)
    out = A.amplfi_inject_whiten(plan, len(par), dev(noise), dev(psd_s), 20.0, 1000.0, approximant=A.SINE_GAUSSIAN,
                                 params=dev(par), gmst=0.7)
    h_det, _ = OP.project(hp_r, hc_r, par, 0.7, dets, n, fs)
    ref = OWH.inject_whiten(noise.astype(np.float64), h_det, psd_s.astype(np.float64) / PSD_SCALE, fs, 20.0, 1000.0)
    assert row_err(out.cpu().numpy().astype(np.float64), ref).max() <= TOL
    h_t, _ = A.amplfi_waveform_td(plan, A.SINE_GAUSSIAN, dev(par), 20.0, 1000.0)
    hp_t, hc_t, _ = OW.waveform_td(OW.SINE_GAUSSIAN, par, n, fs, 20.0, 1000.0)
    got = h_t.cpu().numpy().astype(np.float64)
    assert row_err(got[:, 0], hp_t).max() <= TOL and row_err(got[:, 1], hc_t).max() <= TOL


# ------------------------------------------------------------------------------------------ plans side by side
def test_two_plans_side_by_side_and_plan_reuse():
    """Two plans of different lengths alive at once (they share the device-wide twiddle tables), one of them reused for
    another batch size, approximant and mode: results equal those of fresh plans bit for bit."""
    par16, noise16, psd16 = _make_inputs(16384, 2048.0, 4, [0, 1], 4242)
    par8, noise8, psd8 = _make_inputs(8192, 2048.0, 3, [0, 1], 4243)
    s16, s8 = dev((psd16 * PSD_SCALE).astype(np.float32)), dev((psd8 * PSD_SCALE).astype(np.float32))

    def run(plan, par, noise, psd_s, batch, approx):
        return A.amplfi_inject_whiten(plan, batch, dev(noise[:batch]), psd_s, 20.0, 1000.0, approximant=approx, params=dev(par[:batch]))

    fresh16 = run(A.Plan(16384, 2048.0, [0, 1], 4), par16, noise16, s16, 4, A.IMRPHENOMD)
    fresh8 = run(A.Plan(8192, 2048.0, [0, 1], 3), par8, noise8, s8, 3, A.TAYLORF2)
    fresh16b = run(A.Plan(16384, 2048.0, [0, 1], 4), par16, noise16, s16, 2, A.TAYLORF2)
    pa, pb = A.Plan(16384, 2048.0, [0, 1], 4), A.Plan(8192, 2048.0, [0, 1], 3)
    a1 = run(pa, par16, noise16, s16, 4, A.IMRPHENOMD)
    b1 = run(pb, par8, noise8, s8, 3, A.TAYLORF2)
    a2 = run(pa, par16, noise16, s16, 2, A.TAYLORF2)            # same plan, smaller batch, other approximant
    a3 = run(pa, par16, noise16, s16, 4, A.IMRPHENOMD)          # and back
    torch.cuda.synchronize()
    assert torch.equal(a1, fresh16) and torch.equal(b1, fresh8) and torch.equal(a2, fresh16b) and torch.equal(a3, fresh16)


# ------------------------------------------------------------------------------------------ bench.py's own call at full size
def test_full_size_assemble_batch_and_views_sampled_rows():
    """BASELINE configs[2] at full size through the call bench.py times (amplfi_assemble_batch: strided background window of
    the strip, PSD chain on the plan's side stream), plus the two-view call on the same inputs; sampled rows against the
    oracle, every row finite."""
    wl = WL.make_c2(batch=2048, strip_len=1 << 24)
    B = wl.batch
    plan = A.Plan(wl.n, wl.fs, wl.det_ids, B, nperseg=wl.nperseg)
    strip = dev(wl.strip)
    o, nb = wl.extra["bg_offset"], wl.extra["n_bg"]
    params, offsets = dev(wl.params), dev(wl.offsets)
    out, psd = A.amplfi_assemble_batch(plan, B, strip[:, o:o + nb], strip, params, wl.f_lo, wl.f_hi, offsets=offsets,
                                       approximant=wl.approximant, gmst=wl.gmst)
    t_shift = np.random.Generator(np.random.Philox(3)).uniform(0.0, 1.0, B)
    v1, v2 = A.amplfi_inject_whiten_views(plan, B, strip, psd, wl.f_lo, wl.f_hi, params, dev(t_shift), offsets=offsets,
                                          approximant=wl.approximant, gmst=wl.gmst)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all()) and bool(torch.isfinite(v1).all()) and bool(torch.isfinite(v2).all())
    rows = np.random.default_rng(1).choice(B, size=4, replace=False)
    psd_ref = OWE.welch(wl.strip[:, o:o + nb].astype(np.float64), wl.fs, wl.nperseg)
    assert np.abs(psd.cpu().numpy().astype(np.float64) / PSD_SCALE / psd_ref - 1)[:, 41:2001].max() <= TOL
    noise = OWH.gather(wl.strip, wl.offsets[rows], wl.n)
    d, d2 = OV.two_views(wl.approximant, wl.params[rows], t_shift[rows], noise, psd_ref, wl.gmst, wl.det_ids, wl.fs,
                         wl.f_lo, wl.f_hi)
    idx = torch.from_numpy(rows).to(out.device)
    assert row_err(out[idx].cpu().numpy().astype(np.float64), d).max() <= TOL
    assert row_err(v1[idx].cpu().numpy().astype(np.float64), d).max() <= TOL
    assert row_err(v2[idx].cpu().numpy().astype(np.float64), d2).max() <= TOL
