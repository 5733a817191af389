"""Shared test helpers (input construction only; no method arithmetic)."""
import numpy as np

from paper_2606_18588_b200 import scenes

SH0 = scenes.SH0


def simple_camera(size=32, f=100.0):
    return scenes.Camera(np.eye(3, dtype=np.float32), np.zeros(3, np.float32), f, f, size / 2.0,
                         size / 2.0, size, size)


def gaussians(mean, scale, quat, logit, colour):
    """Degree-0 Gaussians from plain lists."""
    n = len(mean)
    sh = np.zeros((n, 16, 3))
    sh[:, 0, :] = (np.asarray(colour, np.float64) - 0.5) / SH0
    scale = np.asarray(scale, np.float64)
    if scale.ndim == 1:
        scale = np.repeat(scale[:, None], 3, 1)
    return dict(mean=np.asarray(mean, np.float64), log_scale=np.log(scale),
                quat=np.asarray(quat, np.float64), opacity_logit=np.asarray(logit, np.float64), sh=sh)


def random_scene(rng, n, size=32, f=40.0, sh_degree=3, zlo=2.0, zhi=6.0, spread=1.2, ls=-1.6):
    """Tiny random scene in the camera frame of a rotated camera (so W != I)."""
    mean = np.stack([rng.uniform(-spread, spread, n), rng.uniform(-spread, spread, n),
                     rng.uniform(zlo, zhi, n)], 1)
    q = rng.standard_normal((n, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    q *= rng.uniform(0.5, 2.0, (n, 1))  # un-normalised on purpose
    p = dict(mean=mean, log_scale=rng.normal(ls, 0.3, (n, 3)), quat=q,
             opacity_logit=rng.normal(0.5, 1.0, n), sh=rng.normal(0, 0.3, (n, 16, 3)))
    p["sh"][:, 0, :] += 1.0
    # a non-trivial world->camera transform: rotate the world, move the means accordingly
    ang = rng.uniform(-0.4, 0.4, 3)
    cx, sx = np.cos(ang[0]), np.sin(ang[0]); cy, sy = np.cos(ang[1]), np.sin(ang[1]); cz, sz = np.cos(ang[2]), np.sin(ang[2])
    Rx = np.array([[1, 0, 0], [0, cx, -sx], [0, sx, cx]]); Ry = np.array([[cy, 0, sy], [0, 1, 0], [-sy, 0, cy]])
    Rz = np.array([[cz, -sz, 0], [sz, cz, 0], [0, 0, 1]])
    R = Rz @ Ry @ Rx
    t = rng.uniform(-0.5, 0.5, 3)
    # world mean such that R @ mean_w + t == mean (camera frame)
    p["mean"] = (mean - t) @ R  # = R^T (mean - t)
    cam = scenes.Camera(R, t, f, f * 1.1, size / 2.0 + 0.3, size / 2.0 - 0.2, size, size)
    return p, cam


def cam64(cam):
    """Full-precision packing for finite differences (no fp32 rounding of R, t)."""
    a = np.zeros(19)
    a[0:9] = np.asarray(cam.R, np.float64).reshape(9); a[9:12] = np.asarray(cam.t, np.float64)
    a[12:16] = (cam.fx, cam.fy, cam.cx, cam.cy); a[16:19] = (cam.width, cam.height, cam.near_z)
    return a
