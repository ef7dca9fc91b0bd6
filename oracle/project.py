"""Oracle detector projection ("antenna response ... on-the-fly"; Table 1
PAPER.md:138-141 for the sky/polarisation angles).  The paper prints no formula; DESIGN.md
readings R-P1..R-P5.  fp64.
"""
import numpy as np

from .constants import C_SI, DETECTORS


def detector_tensor(xarm, yarm):
    """D = (x x^T - y y^T) / 2 for arm unit vectors x, y."""
    xarm = np.asarray(xarm, dtype=np.float64)
    yarm = np.asarray(yarm, dtype=np.float64)
    return 0.5 * (np.outer(xarm, xarm) - np.outer(yarm, yarm))


def response(ra, dec, psi, gmst, r, xarm, yarm):
    """(F+, Fx, dt) of one detector (vertex r [m], arms xarm, yarm) for a source at (ra, dec),
    polarisation angle psi, Greenwich sidereal angle gmst.

    R-P1: Greenwich hour angle gha = gmst - ra.
    R-P2: X = (-cos psi sin gha - sin psi cos gha sin dec, -cos psi cos gha + sin psi sin gha sin dec,
               sin psi cos dec),
          Y = ( sin psi sin gha - cos psi cos gha sin dec,  sin psi cos gha + cos psi sin gha sin dec,
               cos psi cos dec);   F+ = X.D.X - Y.D.Y,  Fx = X.D.Y + Y.D.X.
    R-P4: n = (cos dec cos gha, -cos dec sin gha, sin dec) points to the source; dt = -(r.n)/c is the
          arrival time at the detector minus the arrival time at the geocentre.
    """
    gha = gmst - ra
    cg, sg = np.cos(gha), np.sin(gha)
    cd, sd = np.cos(dec), np.sin(dec)
    cp, sp = np.cos(psi), np.sin(psi)
    xv = np.array([-cp * sg - sp * cg * sd, -cp * cg + sp * sg * sd, sp * cd])
    yv = np.array([sp * sg - cp * cg * sd, sp * cg + cp * sg * sd, cp * cd])
    nv = np.array([cd * cg, -cd * sg, sd])
    dten = detector_tensor(xarm, yarm)
    fplus = xv @ dten @ xv - yv @ dten @ yv
    fcross = xv @ dten @ yv + yv @ dten @ xv
    dt = -float(np.dot(np.asarray(r, dtype=np.float64), nv)) / C_SI
    return fplus, fcross, dt


def responses(params, gmst, det_ids):
    """[B, D, 3] array of (F+, Fx, dt); params rows as in oracle.waveform (ra, dec, psi = 8, 9, 10)."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    out = np.zeros((params.shape[0], len(det_ids), 3))
    for b, p in enumerate(params):
        for j, d in enumerate(det_ids):
            det = DETECTORS[int(d)]
            out[b, j] = response(p[8], p[9], p[10], gmst, det["r"], det["x"], det["y"])
    return out


def project(hp, hc, params, gmst, det_ids, n, fs):
    """h_d(f_k) = (F+ h+ + Fx hx) * exp(-2 pi i f_k dt_d)   (R-P5), f_k = k fs / n.
    hp, hc: [B, K] complex.  Returns (h_det [B, D, K] complex128, resp [B, D, 3])."""
    hp = np.asarray(hp, dtype=np.complex128)
    hc = np.asarray(hc, dtype=np.complex128)
    resp = responses(params, gmst, det_ids)
    f = np.arange(n // 2 + 1) * (fs / n)
    out = np.zeros((hp.shape[0], len(det_ids), hp.shape[1]), dtype=np.complex128)
    for b in range(hp.shape[0]):
        for j in range(len(det_ids)):
            fp, fc, dt = resp[b, j]
            out[b, j] = (fp * hp[b] + fc * hc[b]) * np.exp(-2j * np.pi * f * dt)
    return out, resp
