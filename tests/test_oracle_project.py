"""Pins for oracle O1 (projection): closed forms, library routines, brute force.
PAPER.md L76 (Sigma = R S S^T R^T), L80 (Sigma2D = J W Sigma W^T J^T)."""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle
from tests.common import SH0, cam64, gaussians, random_scene, simple_camera


def _proj(p, cam, deg=0, cfg=oracle.DEFAULT_CFG):
    return oracle.project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], deg,
                          cam64(cam), cfg)


def _cov_from_conic(co):
    Q = np.array([[co[0], co[1]], [co[1], co[2]]])
    return np.linalg.inv(Q)


def test_on_axis_isotropic_closed_form():
    # Sigma2D = (f s / z)^2 I + 0.3 I for any rotation; radius = ceil(3 sqrt(.))
    cam = simple_camera(32, 100.0)
    rng = np.random.default_rng(0)
    for s, z in [(0.1, 4.0), (0.2, 8.0), (0.05, 2.5)]:
        q = rng.standard_normal(4)
        p = gaussians([[0, 0, z]], [s], [q], [0.0], [[0.9, 0.1, 0.1]])
        pr = _proj(p, cam)
        var = (100.0 * s / z) ** 2 + 0.3
        assert np.allclose(_cov_from_conic(pr.conic_opacity[0]), var * np.eye(2), rtol=1e-12)
        assert pr.radius[0] == math.ceil(3 * math.sqrt(var))
        assert np.allclose(pr.means2d[0], [16.0, 16.0]) and pr.depth[0] == z
        assert abs(pr.conic_opacity[0, 3] - 0.5) < 1e-15  # sigmoid(0)


def test_identity_quat_anisotropic_and_z_rotation():
    # q = identity -> Sigma = diag(s^2): on-axis Sigma2D = diag((f sx/z)^2, (f sy/z)^2) + 0.3.
    # q = rotation by psi about z (w = cos psi/2, z = sin psi/2) rotates the xy block by psi.
    cam = simple_camera(64, 80.0)
    s = np.array([[0.3, 0.1, 0.05]]); z = 5.0
    p = gaussians([[0, 0, z]], s, [[1, 0, 0, 0]], [0.0], [[0.5, 0.5, 0.5]])
    cov = _cov_from_conic(_proj(p, cam).conic_opacity[0])
    assert np.allclose(cov, np.diag([(80 * 0.3 / z) ** 2 + 0.3, (80 * 0.1 / z) ** 2 + 0.3]), rtol=1e-12)
    psi = 0.7
    p["quat"] = np.array([[math.cos(psi / 2), 0, 0, math.sin(psi / 2)]])
    cov = _cov_from_conic(_proj(p, cam).conic_opacity[0])
    Rz = np.array([[math.cos(psi), -math.sin(psi)], [math.sin(psi), math.cos(psi)]])
    expect = Rz @ np.diag([(80 * 0.3 / z) ** 2, (80 * 0.1 / z) ** 2]) @ Rz.T + 0.3 * np.eye(2)
    assert np.allclose(cov, expect, rtol=1e-12)
    # rotation by 90 deg about x maps the y axis onto z: the screen sees (sx, sz)
    p["quat"] = np.array([[math.cos(math.pi / 4), math.sin(math.pi / 4), 0, 0]])
    cov = _cov_from_conic(_proj(p, cam).conic_opacity[0])
    assert np.allclose(cov, np.diag([(80 * 0.3 / z) ** 2 + 0.3, (80 * 0.05 / z) ** 2 + 0.3]), rtol=1e-12)


def test_quaternion_sign_and_scale_invariance():
    rng = np.random.default_rng(1)
    p, cam = random_scene(rng, 16)
    a = _proj(p, cam, 3)
    for c in (-1.0, 3.7):
        p2 = dict(p); p2["quat"] = p["quat"] * c
        b = _proj(p2, cam, 3)
        assert np.allclose(a.conic_opacity, b.conic_opacity, rtol=1e-11)
        assert (a.radius == b.radius).all()


def test_sigma_matches_scipy_rotation():
    # library pin of the quaternion convention: Sigma = Rm diag(s^2) Rm^T with scipy's matrix
    from scipy.spatial.transform import Rotation
    rng = np.random.default_rng(2)
    p, cam = random_scene(rng, 12)
    pr = _proj(p, cam, 0)
    R = np.asarray(cam.R, np.float64); t = np.asarray(cam.t, np.float64)
    for i in range(12):
        if pr.radius[i] == 0:
            continue
        q = p["quat"][i] / np.linalg.norm(p["quat"][i])
        Rm = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()  # scipy is (x,y,z,w)
        Sig = Rm @ np.diag(np.exp(2 * p["log_scale"][i])) @ Rm.T
        pc = R @ p["mean"][i] + t
        # numerical Jacobian of (x,y,z) -> (fx x/z, fy y/z) at pc (inside the clamp region here)
        def pi(v):
            return np.array([cam.fx * v[0] / v[2], cam.fy * v[1] / v[2]])
        h = 1e-6
        J = np.stack([(pi(pc + h * e) - pi(pc - h * e)) / (2 * h) for e in np.eye(3)], 1)
        cov = J @ R @ Sig @ R.T @ J.T + 0.3 * np.eye(2)
        assert np.allclose(_cov_from_conic(pr.conic_opacity[i]), cov, rtol=1e-6)
        lam = np.linalg.eigvalsh(cov)[-1]
        assert pr.radius[i] == math.ceil(3 * math.sqrt(lam))
        assert np.allclose(pr.means2d[i], pi(pc) + [cam.cx, cam.cy], rtol=1e-12)
        assert pr.depth[i] == pytest.approx(pc[2], rel=1e-14)


def test_jacobian_clamp_far_off_axis():
    # x/z beyond 1.3 tan(fov/2): J is evaluated at the clamped point (reading s9), the 2-D mean is not
    cam = simple_camera(32, 100.0)
    lim = 1.3 * 32 / 200.0
    z = 4.0; x = 2.0  # x/z = 0.5 > lim = 0.208
    s = 0.5
    p = gaussians([[x, 0, z]], [s], [[1, 0, 0, 0]], [0.0], [[0.5, 0.5, 0.5]])
    pr = _proj(p, cam)
    tx = lim * z
    J = np.array([[100 / z, 0, -100 * tx / z ** 2], [0, 100 / z, 0]])
    cov = J @ (s * s * np.eye(3)) @ J.T + 0.3 * np.eye(2)
    assert pr.radius[0] > 0
    assert np.allclose(_cov_from_conic(pr.conic_opacity[0]), cov, rtol=1e-12)
    assert pr.means2d[0, 0] == pytest.approx(100 * x / z + 16)


def test_culling():
    cam = simple_camera(32, 100.0)
    p = gaussians([[0, 0, 0.2], [0, 0, -3.0], [0, 0, 0.21], [500.0, 0, 4.0]], [0.01, 0.1, 0.01, 0.1],
                  [[1, 0, 0, 0]] * 4, [0.0] * 4, [[0.5, 0.5, 0.5]] * 4)
    pr = _proj(p, cam)
    assert list(pr.radius > 0) == [False, False, True, False]  # z<=near, behind, kept, off-screen
    assert pr.tiles_touched[0] == 0 and pr.tiles_touched[3] == 0
    assert not pr.conic_opacity[0].any() and not pr.means2d[3].any()


def test_tile_rect_brute_force():
    # independent statement in exact arithmetic: with lo = u-0.5-r, hi = u-0.5+r (pixel-index
    # space), tile column tx is listed iff one of its 16 pixel columns is > lo-1 and one is <= hi-1
    rng = np.random.default_rng(3)
    p, cam = random_scene(rng, 200, size=70, f=60.0)
    pr = _proj(p, cam, 0)
    W = H = 70; TX = TY = 5
    assert (pr.radius > 0).sum() > 50
    for i in np.nonzero(pr.radius > 0)[0]:
        u = Fraction(float(np.float32(pr.means2d[i, 0]))); v = Fraction(float(np.float32(pr.means2d[i, 1])))
        r = int(pr.radius[i])
        def cover(c, ntiles):
            lo, hi = c - Fraction(1, 2) - r, c - Fraction(1, 2) + r
            out = []
            for t in range(ntiles):
                cols = range(16 * t, 16 * t + 16)
                if any(cc > lo - 1 for cc in cols) and any(cc <= hi - 1 for cc in cols):
                    out.append(t)
            return out
        xs, ys = cover(u, TX), cover(v, TY)
        x0, y0, x1, y1 = pr.rect[i]
        assert list(range(x0, x1)) == xs and list(range(y0, y1)) == ys
        assert pr.tiles_touched[i] == len(xs) * len(ys)


def test_sh_orthonormal_by_quadrature():
    # int Y_i Y_j dOmega = delta_ij  (Gauss-Legendre in cos(theta) x uniform phi)
    nt, nph = 16, 32
    xs, ws = np.polynomial.legendre.leggauss(nt)
    G = np.zeros((16, 16))
    for ct, w in zip(xs, ws):
        st = math.sqrt(1 - ct * ct)
        for k in range(nph):
            ph = 2 * math.pi * k / nph
            Y = oracle.sh_basis(3, [st * math.cos(ph), st * math.sin(ph), ct])
            G += w * (2 * math.pi / nph) * np.outer(Y, Y)
    assert np.abs(G - np.eye(16)).max() < 1e-12


def test_sh_matches_scipy_complex_harmonics():
    # library pin: index l(l+1)+m; m>0: sqrt2 Re Y_l^m, m<0: sqrt2 Im Y_l^|m|, with scipy's
    # Condon-Shortley phase kept (this is the sign convention of reading s13)
    import scipy.special as sp
    rng = np.random.default_rng(4)
    for _ in range(10):
        d = rng.standard_normal(3); d /= np.linalg.norm(d)
        theta = math.acos(d[2]); phi = math.atan2(d[1], d[0])
        Y = oracle.sh_basis(3, d)
        for l in range(4):
            for m in range(-l, l + 1):
                if hasattr(sp, "sph_harm_y"):
                    c = sp.sph_harm_y(l, abs(m), theta, phi)
                else:
                    c = sp.sph_harm(abs(m), l, phi, theta)
                ref = c.real if m == 0 else (math.sqrt(2) * c.real if m > 0 else math.sqrt(2) * c.imag)
                assert Y[l * (l + 1) + m] == pytest.approx(ref, abs=1e-13)


def test_colour_degree0_closed_form_and_clamp():
    cam = simple_camera(32, 100.0)
    p = gaussians([[0.1, -0.2, 3.0]] * 2, [0.1, 0.1], [[1, 0, 0, 0]] * 2, [1.0, -1.0],
                  [[0.9, 0.1, 0.25], [0.2, 0.2, 0.2]])
    p["sh"][1, 0, :] = [-3.0, 0.4, -2.0]
    pr = _proj(p, cam)
    assert np.allclose(pr.rgb[0], [0.9, 0.1, 0.25], atol=1e-12)
    assert np.allclose(pr.rgb[1], [0.0, 0.5 + SH0 * 0.4, 0.0], atol=1e-12)
    assert pr.clamp[0] == 0 and pr.clamp[1] == 0b101
    assert pr.conic_opacity[0, 3] == pytest.approx(1 / (1 + math.exp(-1.0)))


def test_colour_view_dependence_uses_direction_from_camera_centre():
    # degree 1: rgb = 0.5 + Y0 sh0 - k1 y sh1 + k1 z sh2 - k1 x sh3, dir = (mu - o)/|mu - o|
    rng = np.random.default_rng(5)
    p, cam = random_scene(rng, 8)
    pr = _proj(p, cam, 1)
    R = np.asarray(cam.R, np.float64); t = np.asarray(cam.t, np.float64)
    o = -R.T @ t
    k1 = math.sqrt(3 / (4 * math.pi))
    for i in range(8):
        if pr.radius[i] == 0:
            continue
        d = p["mean"][i] - o; d /= np.linalg.norm(d)
        ref = 0.5 + SH0 * p["sh"][i, 0] - k1 * d[1] * p["sh"][i, 1] + k1 * d[2] * p["sh"][i, 2] - k1 * d[0] * p["sh"][i, 3]
        assert np.allclose(pr.rgb[i], np.maximum(ref, 0), atol=1e-12)
