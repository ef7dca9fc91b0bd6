"""Pins for oracle.project (P-1..P-5; BASELINE north_star checks
"F+^2+Fx^2 independent of the polarisation angle", "inter-site delays never exceed the
light-travel time")."""
import itertools

import numpy as np
import pytest

from oracle import constants as C
from oracle import project as P

from conftest import read_golden

G = read_golden("antenna_worked_example.txt")


def test_worked_example_values():
    for d, name in ((0, "H1"), (1, "L1"), (2, "V1")):
        det = C.DETECTORS[d]
        got = P.response(1.0, 0.5, 0.7, 2.0, det["r"], det["x"], det["y"])
        assert np.abs(np.array(got) - np.array(G[name])).max() < 5e-12


def test_site_geometry_self_consistent():
    # P-3: unit arms, orthogonal arms, baselines equal the published light-travel times
    for d in range(3):
        det = C.DETECTORS[d]
        assert abs(np.linalg.norm(det["x"]) - 1) < 1e-10 and abs(np.linalg.norm(det["y"]) - 1) < 1e-10
        assert abs(np.dot(det["x"], det["y"])) < 2e-5
        # arms are (nearly) horizontal: perpendicular to the local vertical within 0.5 deg
        up = det["r"] / np.linalg.norm(det["r"])
        assert abs(np.dot(det["x"], up)) < 0.01 and abs(np.dot(det["y"], up)) < 0.01
        assert 6.35e6 < np.linalg.norm(det["r"]) < 6.38e6
    pairs = [(0, 1), (0, 2), (1, 2)]
    for (i, j), ms in zip(pairs, G["baselines_ms"]):
        base = np.linalg.norm(C.DETECTORS[i]["r"] - C.DETECTORS[j]["r"]) / C.C_SI * 1e3
        assert abs(base - ms) < 1e-4
    # published values 10.0 / 27.3 / 26.4 ms
    assert np.allclose(G["baselines_ms"], [10.0, 27.3, 26.4], atol=0.06)


def test_psi_independence_and_bounds():
    rng = np.random.default_rng(5)
    for _ in range(50):
        ra, dec, gmst = rng.uniform(0, 2 * np.pi), np.arcsin(rng.uniform(-1, 1)), rng.uniform(0, 2 * np.pi)
        for d in range(3):
            det = C.DETECTORS[d]
            tot = []
            for psi in np.linspace(0, np.pi, 13):
                fp, fc, dt = P.response(ra, dec, psi, gmst, det["r"], det["x"], det["y"])
                tot.append(fp * fp + fc * fc)
                fp2, fc2, dt2 = P.response(ra, dec, psi + np.pi / 2, gmst, det["r"], det["x"], det["y"])
                assert abs(fp + fp2) < 1e-14 and abs(fc + fc2) < 1e-14 and dt == dt2
            assert np.ptp(tot) < 1e-14 and max(tot) <= 1 + 1e-9
            assert abs(dt) <= np.linalg.norm(det["r"]) / C.C_SI + 1e-12 and abs(dt) < 0.0213


def test_depends_on_gmst_minus_ra_only():
    det = C.DETECTORS[1]
    a = P.response(0.3, -0.2, 0.4, 1.1, det["r"], det["x"], det["y"])
    b = P.response(0.3 + 0.77, -0.2, 0.4, 1.1 + 0.77, det["r"], det["x"], det["y"])
    assert np.allclose(a, b, atol=1e-14)


def test_inter_site_delay_bounded_by_light_travel_time():
    rng = np.random.default_rng(6)
    p = np.zeros((200, 11))
    p[:, 8] = rng.uniform(0, 2 * np.pi, 200)
    p[:, 9] = np.arcsin(rng.uniform(-1, 1, 200))
    r = P.responses(p, 0.3, [0, 1, 2])
    for i, j in itertools.combinations(range(3), 2):
        lim = np.linalg.norm(C.DETECTORS[i]["r"] - C.DETECTORS[j]["r"]) / C.C_SI
        assert np.all(np.abs(r[:, i, 2] - r[:, j, 2]) <= lim + 1e-12)


def test_overhead_source_unit_response_and_textbook_pattern():
    # A detector at the north pole with arms along x, y: the textbook pattern is
    # F+ = (1+cos^2 th)/2 cos 2ph cos 2psi - cos th sin 2ph sin 2psi (up to the psi origin/sign),
    # Fx = (1+cos^2 th)/2 cos 2ph sin 2psi + cos th sin 2ph cos 2psi.  Compare rotation-invariant content:
    # F+^2 + Fx^2 = ((1+cos^2 th)/2)^2 cos^2 2ph + cos^2 th sin^2 2ph.
    r, xa, ya = np.array([0, 0, 6.37e6]), np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    rng = np.random.default_rng(9)
    for _ in range(20):
        th, ph, psi = np.arccos(rng.uniform(-1, 1)), rng.uniform(0, 2 * np.pi), rng.uniform(0, np.pi)
        dec, gha = np.pi / 2 - th, -ph          # n = (cos dec cos gha, -cos dec sin gha, sin dec) = (sin th cos ph, sin th sin ph, cos th)
        fp, fc, dt = P.response(-gha, dec, psi, 0.0, r, xa, ya)
        want = (0.5 * (1 + np.cos(th) ** 2)) ** 2 * np.cos(2 * ph) ** 2 + np.cos(th) ** 2 * np.sin(2 * ph) ** 2
        assert abs(fp * fp + fc * fc - want) < 1e-13
        assert abs(dt + 6.37e6 * np.cos(th) / C.C_SI) < 1e-15       # wave reaches a detector nearer the source earlier
    fp, fc, _ = P.response(0.0, np.pi / 2, 0.0, 0.0, r, xa, ya)
    assert abs(fp * fp + fc * fc - 1) < 1e-14
    # real site: overhead of H1 the response is 1
    up = C.DETECTORS[0]["x"]
    n = np.cross(C.DETECTORS[0]["x"], C.DETECTORS[0]["y"])
    n /= np.linalg.norm(n)
    dec, gha = np.arcsin(n[2]), np.arctan2(-n[1], n[0])
    fp, fc, _ = P.response(-gha, dec, 0.3, 0.0, C.DETECTORS[0]["r"], C.DETECTORS[0]["x"], C.DETECTORS[0]["y"])
    assert abs(fp * fp + fc * fc - 1) < 1e-6


def test_xy_handedness():
    # X x Y = -n (P-2)
    ra, dec, psi, gmst = 0.4, -0.7, 1.2, 2.2
    gha = gmst - ra
    cg, sg, cd, sd, cp, sp = np.cos(gha), np.sin(gha), np.cos(dec), np.sin(dec), np.cos(psi), np.sin(psi)
    xv = np.array([-cp * sg - sp * cg * sd, -cp * cg + sp * sg * sd, sp * cd])
    yv = np.array([sp * sg - cp * cg * sd, sp * cg + cp * sg * sd, cp * cd])
    nv = np.array([cd * cg, -cd * sg, sd])
    assert np.allclose(np.cross(xv, yv), -nv, atol=1e-15)
    # the oracle's F+ equals the contraction with e+ = XX - YY built here
    det = C.DETECTORS[2]
    dten = 0.5 * (np.outer(det["x"], det["x"]) - np.outer(det["y"], det["y"]))
    fp, fc, _ = P.response(ra, dec, psi, gmst, det["r"], det["x"], det["y"])
    assert abs(fp - np.sum(dten * (np.outer(xv, xv) - np.outer(yv, yv)))) < 1e-15
    assert abs(fc - np.sum(dten * (np.outer(xv, yv) + np.outer(yv, xv)))) < 1e-15


def test_one_sample_delay_is_circular_roll():
    # P-5: multiplying by exp(-2 pi i f dt) with dt = 1/fs equals np.roll(x, 1)
    n, fs = 256, 256.0
    x = np.random.default_rng(2).standard_normal(n)
    xk = np.fft.rfft(x)
    f = np.arange(n // 2 + 1) * fs / n
    y = np.fft.irfft(xk * np.exp(-2j * np.pi * f / fs), n)
    assert np.abs(y - np.roll(x, 1)).max() < 1e-12


def test_project_combines_polarisations_and_delay():
    rng = np.random.default_rng(3)
    k = 65
    hp = rng.standard_normal((2, k)) + 1j * rng.standard_normal((2, k))
    hc = rng.standard_normal((2, k)) + 1j * rng.standard_normal((2, k))
    p = np.zeros((2, 11))
    p[:, 8:11] = [[1.0, 0.5, 0.7], [2.0, -0.3, 0.1]]
    h, resp = P.project(hp, hc, p, 2.0, [0, 2], 128, 128.0)
    assert h.shape == (2, 2, k)
    b, j, kk = 1, 1, 17
    want = (resp[b, j, 0] * hp[b, kk] + resp[b, j, 1] * hc[b, kk]) * np.exp(-2j * np.pi * kk * 1.0 * resp[b, j, 2])
    assert abs(h[b, j, kk] - want) < 1e-14
    assert np.abs(np.array(G["V1"]) - resp[0, 1]).max() < 5e-12
