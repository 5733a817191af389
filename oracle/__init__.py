"""CPU oracle for the Splaxel hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes binding of ``oracle/splx_oracle.cpp`` (plain single-threaded C++, fp64)
plus a small driver that chains the stages the way SURVEY.md s3(b) does.  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` leg may import this package.  It shares no code with the
CUDA path and never imports ``paper_2606_18588_b200``.

Every function cites the passage of PAPER.md it follows in the C++ source.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "splx_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

TILE = 16
#: alpha_min, alpha_max, T_eps, dilation, lim_factor, radius_floor (readings s2, s9)
DEFAULT_CFG = (1.0 / 255.0, 0.99, 1e-4, 0.3, 1.3, 0.1)
#: smooth mode for finite differences: no alpha skip, no clamp, no early exit
SMOOTH_CFG = (0.0, 1.0, 0.0, 0.3, 1.3, 0.1)


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", _LIB, _SRC]
        subprocess.check_call(cmd)
    from . import dssim as _dssim      # the D-SSIM term has its own plain-C file
    _dssim.build(force)
    return _LIB


def _c(arr, dtype):
    a = np.ascontiguousarray(arr, dtype=dtype)
    return a


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        L.orc_count_tiles.restype = ctypes.c_uint64
        L.orc_render_partial.restype = ctypes.c_uint64
        L.orc_l1.restype = ctypes.c_double
        _lib = L
    return _lib


def make_camera(R, t, fx, fy, cx, cy, width, height, near_z=0.2) -> np.ndarray:
    """Pack a pinhole camera: p_cam = R @ mean + t (row-major R)."""
    cam = np.zeros(19, dtype=np.float64)
    cam[0:9] = np.asarray(R, dtype=np.float64).reshape(9)
    cam[9:12] = np.asarray(t, dtype=np.float64).reshape(3)
    cam[12:16] = (fx, fy, cx, cy)
    cam[16:19] = (width, height, near_z)
    return cam


def cam_wh(cam):
    return int(cam[16]), int(cam[17])


def tiles_xy(W, H):
    return (W + TILE - 1) // TILE, (H + TILE - 1) // TILE


@dataclass
class Projected:
    means2d: np.ndarray
    depth: np.ndarray
    conic_opacity: np.ndarray
    rgb: np.ndarray
    radius: np.ndarray
    tiles_touched: np.ndarray
    clamp: np.ndarray
    rect: np.ndarray | None = None
    radius_margin: np.ndarray | None = None


@dataclass
class Binning:
    offsets: np.ndarray
    keys: np.ndarray
    vals: np.ndarray
    ranges: np.ndarray
    M: int


@dataclass
class Partial:
    ct: np.ndarray       # [H,W,4] premultiplied rgb, T
    d: np.ndarray        # [H,W]
    n_contrib: np.ndarray
    margin: np.ndarray | None = None
    t_exit: np.ndarray | None = None
    walked: int = 0


def project(mean, log_scale, quat, opacity_logit, sh, sh_degree, cam, cfg=DEFAULT_CFG) -> Projected:
    n = int(np.asarray(mean).shape[0])
    mean = _c(mean, np.float64).reshape(n, 3)
    log_scale = _c(log_scale, np.float64).reshape(n, 3)
    quat = _c(quat, np.float64).reshape(n, 4)
    opacity_logit = _c(opacity_logit, np.float64).reshape(n)
    sh = _c(sh, np.float64).reshape(n, 16, 3)
    cam = _c(cam, np.float64); cfg = _c(cfg, np.float64)
    out = Projected(np.zeros((n, 2)), np.zeros(n), np.zeros((n, 4)), np.zeros((n, 3)),
                    np.zeros(n, np.int32), np.zeros(n, np.uint32), np.zeros(n, np.uint8),
                    np.zeros((n, 4), np.int32), np.zeros(n))
    lib().orc_project(ctypes.c_int64(n), _p(mean), _p(log_scale), _p(quat), _p(opacity_logit),
                      _p(sh), ctypes.c_int(sh_degree), _p(cam), _p(cfg), _p(out.means2d),
                      _p(out.depth), _p(out.conic_opacity), _p(out.rgb), _p(out.radius),
                      _p(out.tiles_touched), _p(out.clamp), _p(out.rect), _p(out.radius_margin))
    return out


def depth_key(mean, cam):
    """The camera depth as the sort key sees it (reading s12): evaluated in fp32 in a fixed operation order, so that the
    oracle and the kernel order near-equal depths alike.  Returned as float64 values that are exact fp32 numbers."""
    n = int(np.asarray(mean).shape[0])
    mean = _c(mean, np.float64).reshape(n, 3)
    cam = _c(cam, np.float64)
    out = np.zeros(n)
    lib().orc_depth_key(ctypes.c_int64(n), _p(mean), _p(cam), _p(out))
    return out


def count_tiles(means2d, radius, W, H):
    n = int(np.asarray(radius).shape[0])
    means2d = _c(means2d, np.float64).reshape(n, 2)
    radius = _c(radius, np.int32)
    tt = np.zeros(n, np.uint32)
    M = lib().orc_count_tiles(ctypes.c_int64(n), _p(means2d), _p(radius), ctypes.c_int(W),
                              ctypes.c_int(H), _p(tt))
    return int(M), tt


def bin_sort(means2d, radius, depth, W, H) -> Binning:
    n = int(np.asarray(radius).shape[0])
    means2d = _c(means2d, np.float64).reshape(n, 2)
    radius = _c(radius, np.int32)
    depth = _c(depth, np.float64).reshape(n)
    M, _ = count_tiles(means2d, radius, W, H)
    TX, TY = tiles_xy(W, H)
    b = Binning(np.zeros(n, np.uint32), np.zeros(M, np.uint64), np.zeros(M, np.uint32),
                np.zeros((TX * TY, 2), np.uint32), M)
    lib().orc_bin_sort(ctypes.c_int64(n), _p(means2d), _p(radius), _p(depth), ctypes.c_int(W),
                       ctypes.c_int(H), _p(b.offsets), _p(b.keys), _p(b.vals), _p(b.ranges))
    return b


def _tiles(tile_list):
    if tile_list is None:
        return None, 0
    tl = _c(tile_list, np.int32)
    return tl, int(tl.shape[0])


def render_partial(means2d, conic_opacity, rgb, depth, vals, ranges, W, H, cfg=DEFAULT_CFG,
                   tile_list=None) -> Partial:
    n = int(np.asarray(depth).shape[0])
    means2d = _c(means2d, np.float64).reshape(n, 2)
    conic_opacity = _c(conic_opacity, np.float64).reshape(n, 4)
    rgb = _c(rgb, np.float64).reshape(n, 3)
    depth = _c(depth, np.float64).reshape(n)
    vals = _c(vals, np.uint32); ranges = _c(ranges, np.uint32)
    cfg = _c(cfg, np.float64)
    tl, nt = _tiles(tile_list)
    out = Partial(np.zeros((H, W, 4)), np.zeros((H, W)), np.zeros((H, W), np.uint32),
                  np.full((H, W), np.inf), np.full((H, W), -1.0))
    out.ct[..., 3] = 1.0
    out.walked = int(lib().orc_render_partial(
        _p(means2d), _p(conic_opacity), _p(rgb), _p(depth), _p(vals), _p(ranges), ctypes.c_int(W),
        ctypes.c_int(H), _p(cfg), _p(tl), ctypes.c_int64(nt), _p(out.ct), _p(out.d),
        _p(out.n_contrib), _p(out.margin), _p(out.t_exit)))
    return out


def compose(ct, d, bg=(0.0, 0.0, 0.0), tile_list=None):
    """ct[K,H,W,4], d[K,H,W] -> image[H,W,3], T_total[H,W], order[H,W,K], order_margin[H,W]."""
    ct = _c(ct, np.float64); d = _c(d, np.float64)
    K, H, W, _ = ct.shape
    bg = _c(bg, np.float64)
    tl, nt = _tiles(tile_list)
    image = np.zeros((H, W, 3)); T_total = np.ones((H, W))
    order = np.zeros((H, W, K), np.int32); om = np.full((H, W), np.inf)
    lib().orc_compose(ctypes.c_int(K), _p(ct), _p(d), ctypes.c_int(W), ctypes.c_int(H), _p(bg),
                      _p(tl), ctypes.c_int64(nt), _p(image), _p(T_total), _p(order), _p(om))
    return image, T_total, order, om


def compose_bwd(ct, d, g_image, bg=(0.0, 0.0, 0.0), g_T_total=None, tile_list=None):
    ct = _c(ct, np.float64); d = _c(d, np.float64)
    K, H, W, _ = ct.shape
    bg = _c(bg, np.float64)
    g_image = _c(g_image, np.float64).reshape(H, W, 3)
    gT = _c(g_T_total, np.float64).reshape(H, W) if g_T_total is not None else None
    tl, nt = _tiles(tile_list)
    g_ct = np.zeros((K, H, W, 4))
    lib().orc_compose_bwd(ctypes.c_int(K), _p(ct), _p(d), ctypes.c_int(W), ctypes.c_int(H), _p(bg),
                          _p(g_image), _p(gT), _p(tl), ctypes.c_int64(nt), _p(g_ct))
    return g_ct


def raster_bwd(means2d, conic_opacity, rgb, vals, ranges, W, H, g_ct, cfg=DEFAULT_CFG,
               tile_list=None):
    """Returns (g_means2d[n,2], g_conic[n,3], g_opacity[n], g_rgb[n,3]) for one partition."""
    n = int(np.asarray(conic_opacity).shape[0])
    means2d = _c(means2d, np.float64).reshape(n, 2)
    conic_opacity = _c(conic_opacity, np.float64).reshape(n, 4)
    rgb = _c(rgb, np.float64).reshape(n, 3)
    vals = _c(vals, np.uint32); ranges = _c(ranges, np.uint32)
    cfg = _c(cfg, np.float64)
    g_ct = _c(g_ct, np.float64).reshape(H, W, 4)
    tl, nt = _tiles(tile_list)
    gm = np.zeros((n, 2)); gc = np.zeros((n, 3)); go = np.zeros(n); gr = np.zeros((n, 3))
    lib().orc_raster_bwd(_p(means2d), _p(conic_opacity), _p(rgb), _p(vals), _p(ranges),
                         ctypes.c_int(W), ctypes.c_int(H), _p(cfg), _p(tl), ctypes.c_int64(nt),
                         _p(g_ct), _p(gm), _p(gc), _p(go), _p(gr))
    return gm, gc, go, gr


def project_bwd(mean, log_scale, quat, opacity_logit, sh, sh_degree, cam, radius, clamp,
                g_means2d, g_conic, g_opacity, g_rgb, cfg=DEFAULT_CFG):
    """Returns dict of parameter gradients for one partition."""
    n = int(np.asarray(mean).shape[0])
    mean = _c(mean, np.float64).reshape(n, 3)
    log_scale = _c(log_scale, np.float64).reshape(n, 3)
    quat = _c(quat, np.float64).reshape(n, 4)
    opacity_logit = _c(opacity_logit, np.float64).reshape(n)
    sh = _c(sh, np.float64).reshape(n, 16, 3)
    cam = _c(cam, np.float64); cfg = _c(cfg, np.float64)
    radius = _c(radius, np.int32); clamp = _c(clamp, np.uint8)
    g_means2d = _c(g_means2d, np.float64); g_conic = _c(g_conic, np.float64)
    g_opacity = _c(g_opacity, np.float64); g_rgb = _c(g_rgb, np.float64)
    g = dict(mean=np.zeros((n, 3)), log_scale=np.zeros((n, 3)), quat=np.zeros((n, 4)),
             opacity_logit=np.zeros(n), sh=np.zeros((n, 16, 3)))
    lib().orc_project_bwd(ctypes.c_int64(n), _p(mean), _p(log_scale), _p(quat), _p(opacity_logit),
                          _p(sh), ctypes.c_int(sh_degree), _p(cam), _p(cfg), _p(radius), _p(clamp),
                          _p(g_means2d), _p(g_conic), _p(g_opacity), _p(g_rgb), _p(g["mean"]),
                          _p(g["log_scale"]), _p(g["quat"]), _p(g["opacity_logit"]), _p(g["sh"]))
    return g


def l1(image, target):
    image = _c(image, np.float64); target = _c(target, np.float64)
    g = np.zeros_like(image)
    L = lib().orc_l1(ctypes.c_int64(image.size), _p(image), _p(target), _p(g))
    return float(L), g


def adam(param, grad, m, v, lr, beta1=0.9, beta2=0.999, eps=1e-15, step=1):
    """In place on float64 arrays param, m, v."""
    assert param.dtype == np.float64 and m.dtype == np.float64 and v.dtype == np.float64
    grad = _c(grad, np.float64)
    lib().orc_adam(ctypes.c_int64(param.size), _p(param), _p(grad), _p(m), _p(v),
                   ctypes.c_double(lr), ctypes.c_double(beta1), ctypes.c_double(beta2),
                   ctypes.c_double(eps), ctypes.c_int(step))


def sh_basis(deg, direction):
    d = _c(direction, np.float64).reshape(3)
    Y = np.zeros(16)
    lib().orc_sh_basis(ctypes.c_int(deg), _p(d), _p(Y))
    return Y


# ---------------------------------------------------------------------------
# Driver: one iteration of SURVEY.md s3(b) on K partitions (K "simulated ranks").
# ---------------------------------------------------------------------------
PARAM_KEYS = ("mean", "log_scale", "quat", "opacity_logit", "sh")


@dataclass
class IterationResult:
    proj: list = field(default_factory=list)       # K Projected
    bins: list = field(default_factory=list)       # K Binning
    partials: list = field(default_factory=list)   # K Partial
    image: np.ndarray | None = None
    T_total: np.ndarray | None = None
    order: np.ndarray | None = None
    order_margin: np.ndarray | None = None
    loss: float = 0.0
    g_image: np.ndarray | None = None
    g_ct: np.ndarray | None = None
    grads2d: list = field(default_factory=list)    # K tuples (gm, gc, go, gr)
    grads: list = field(default_factory=list)      # K dicts
    walked: int = 0


def forward(parts, cam, sh_degree, bg=(0.0, 0.0, 0.0), cfg=DEFAULT_CFG, tile_list=None):
    """parts: list of K dicts with PARAM_KEYS (one partition each)."""
    W, H = cam_wh(cam)
    res = IterationResult()
    for p in parts:
        pr = project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], sh_degree,
                     cam, cfg)
        b = bin_sort(pr.means2d, pr.radius, depth_key(p["mean"], cam), W, H)     # order by the fp32 key (s12)
        pa = render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, b.vals, b.ranges, W, H,
                            cfg, tile_list)
        res.proj.append(pr); res.bins.append(b); res.partials.append(pa)
        res.walked += pa.walked
    ct = np.stack([pa.ct for pa in res.partials]); d = np.stack([pa.d for pa in res.partials])
    res.image, res.T_total, res.order, res.order_margin = compose(ct, d, bg, tile_list)
    return res


def backward(parts, cam, sh_degree, res: IterationResult, g_image, bg=(0.0, 0.0, 0.0),
             cfg=DEFAULT_CFG, tile_list=None, g_T_total=None):
    W, H = cam_wh(cam)
    ct = np.stack([pa.ct for pa in res.partials]); d = np.stack([pa.d for pa in res.partials])
    res.g_image = g_image
    res.g_ct = compose_bwd(ct, d, g_image, bg, g_T_total, tile_list)
    res.grads2d, res.grads = [], []
    for k, p in enumerate(parts):
        pr, b = res.proj[k], res.bins[k]
        g2 = raster_bwd(pr.means2d, pr.conic_opacity, pr.rgb, b.vals, b.ranges, W, H, res.g_ct[k],
                        cfg, tile_list)
        g = project_bwd(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"],
                        sh_degree, cam, pr.radius, pr.clamp, *g2, cfg=cfg)
        res.grads2d.append(g2); res.grads.append(g)
    return res


def iteration(parts, cam, sh_degree, target, bg=(0.0, 0.0, 0.0), cfg=DEFAULT_CFG):
    """forward + L1 + backward (steps a1..a10)."""
    res = forward(parts, cam, sh_degree, bg, cfg)
    res.loss, g_image = l1(res.image, target)
    return backward(parts, cam, sh_degree, res, g_image, bg, cfg)
