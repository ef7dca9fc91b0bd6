"""Oracle for the two data views (d, d') of the self-supervised pre-training (Figure 2: "the same
background strain with a time-shifted signal injected, the parameters of which are otherwise the same ... The
time shift is random up to 1s"; section 4.1: "all signal parameters being the same except the time
of arrival").  SURVEY.md 8(f)-1.  fp64; test infrastructure only.
"""
import numpy as np

from . import project as OP
from . import waveform as OW
from . import whiten as OWH


def two_views(approximant, params, t_shift, noise, psd, gmst, det_ids, fs, f_lo, f_hi):
    """Returns (d, d'): [B, D, N] each.  d is the ordinary injected + whitened batch; d' repeats every step
    with the arrival time t_c replaced by t_c + t_shift[b] (column 7 of params) and everything else -- the
    background segment, the power spectrum, the other ten parameters -- unchanged."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    t_shift = np.asarray(t_shift, dtype=np.float64)
    n = np.asarray(noise).shape[-1]
    views = []
    for shift in (np.zeros_like(t_shift), t_shift):
        p = params.copy()
        p[:, 7] = p[:, 7] + shift
        hp, hc, _ = OW.waveform_fd(approximant, p, n, fs, f_lo, f_hi)
        h_det, _ = OP.project(hp, hc, p, gmst, det_ids, n, fs)
        views.append(OWH.inject_whiten(noise, h_det, psd, fs, f_lo, f_hi))
    return views[0], views[1]
