"""Helpers for the -m gpu parity tests: run the CUDA stages through the C ABI binding and bring
their outputs to the host as numpy arrays; fragile-pixel bookkeeping (DESIGN.md 'Parity
protocol').  No method arithmetic here: the expected values always come from oracle/."""
import numpy as np
import torch

import oracle
from paper_2606_18588_b200 import binding, scenes
from paper_2606_18588_b200.engine import Trainer

#: decisions closer than this (relative) to a threshold may flip between fp32 and fp64
FRAGILE_MARGIN = 1e-5
#: a flipped decision changes a pixel by at most alpha_min * T (skip) or alpha * T_exit < 1e-2 (exit)
FRAGILE_TOL = 1e-2
TOL = 1e-5   # north_star: 1e-5 abs/rel on fp32 images and T
#: north_star: 1e-3 rel on accumulated gradients -- max |g - ref| against the tensor's max |ref| (DESIGN.md s6 'Tolerances')
GRAD_MAX_TOL = 1e-3


def np32(t):
    return t.detach().cpu().numpy()


def u32(t):
    return t.detach().cpu().numpy().view(np.uint32)


def u64(t):
    return t.detach().cpu().numpy().view(np.uint64)


def make_trainer(sc: scenes.Scene, cfg=None, capacity=None, **kw) -> Trainer:
    cam = sc.cameras[0]
    return Trainer(sc.params, sc.part_offsets, cam.width, cam.height, sc.sh_degree, sc.bg, capacity=capacity, cfg=cfg)


def close(a, ref, tol=TOL):
    """|a - ref| <= tol * max(1, |ref|) elementwise -> bool array."""
    ref = np.asarray(ref, np.float64)
    return np.abs(np.asarray(a, np.float64) - ref) <= tol * np.maximum(1.0, np.abs(ref))


def gpu_projected(tr: Trainer):
    p = tr.proj
    return oracle.Projected(np32(p.means2d).astype(np.float64), np32(p.depth).astype(np.float64),
                            np32(p.conic_opacity).astype(np.float64), np32(p.rgb).astype(np.float64),
                            np32(p.radius).copy(), u32(p.tiles_touched).copy(), np32(p.clamp).copy())


def gpu_bins(tr: Trainer):
    """Per partition: (keys with the partition prefix removed, vals local to the partition, ranges)."""
    M = tr.num_intersections()
    keys = u64(tr.bins.keys)[:M]
    vals = u32(tr.bins.vals)[:M]
    ranges = u32(tr.bins.tile_ranges).reshape(tr.K, -1, 2)
    return M, keys, vals, ranges


def oracle_parts_projected(pr: oracle.Projected, part_offsets):
    out = []
    for k in range(len(part_offsets) - 1):
        a, b = int(part_offsets[k]), int(part_offsets[k + 1])
        out.append(oracle.Projected(pr.means2d[a:b], pr.depth[a:b], pr.conic_opacity[a:b], pr.rgb[a:b],
                                    pr.radius[a:b], pr.tiles_touched[a:b], pr.clamp[a:b]))
    return out


def rel_l2(a, ref):
    ref = np.asarray(ref, np.float64)
    den = np.sqrt((ref ** 2).sum())
    return float(np.sqrt(((np.asarray(a, np.float64) - ref) ** 2).sum()) / max(den, 1e-300))


def grad_close(a, ref, tol=1e-3):
    """north_star: 1e-3 rel on accumulated gradients: max abs error against the tensor's max."""
    ref = np.asarray(ref, np.float64)
    scale = max(np.abs(ref).max(), 1e-30)
    return float(np.abs(np.asarray(a, np.float64) - ref).max() / scale)


def fragile_gaussians(res, W, H, alpha_min=1.0 / 255.0):
    """Per partition, the Gaussians that blend (or nearly blend: alpha >= alpha_min / 2) at a FRAGILE pixel of the
    oracle's result `res` (oracle.IterationResult) -- a pixel where a skip / exit decision lies within fp32 rounding of
    its threshold.  A flipped decision changes that pixel's term in the gradient of exactly these Gaussians, so the
    protocol excludes them from the 1e-3 max-error statistic and counts them."""
    TX = (W + 15) // 16
    out = []
    for pr, b, pa in zip(res.proj, res.bins, res.partials):
        mark = np.zeros(pr.radius.shape[0], bool)
        ys, xs = np.nonzero(pa.margin < FRAGILE_MARGIN)
        for y, x in zip(ys, xs):
            a, e = b.ranges[(y // 16) * TX + x // 16]
            idx = b.vals[a:e]
            dx = pr.means2d[idx, 0] - (x + 0.5); dy = pr.means2d[idx, 1] - (y + 0.5)
            co = pr.conic_opacity[idx]
            power = -0.5 * (co[:, 0] * dx * dx + co[:, 2] * dy * dy) - co[:, 1] * dx * dy
            mark[idx[(power <= 0) & (co[:, 3] * np.exp(np.minimum(power, 0)) >= 0.5 * alpha_min)]] = True
        out.append(mark)
    return out


def grad_rows_close(a, ref, width, rtol=1e-3, atol_of_max=1e-5):
    """the max-normalised error is blind to the many small rows.  Per row (Gaussian):
    max|a - ref| <= rtol * max|ref_row| + atol_of_max * max|ref|  (the absolute term is the noise floor of the fp32
    atomic sums: a row's gradient is a sum of up to thousands of terms of the tensor's scale).  Returns the fraction of
    rows that hold it."""
    a = np.asarray(a, np.float64).reshape(-1, width); ref = np.asarray(ref, np.float64).reshape(-1, width)
    err = np.abs(a - ref).max(1)
    return float((err <= rtol * np.abs(ref).max(1) + atol_of_max * max(np.abs(ref).max(), 1e-300)).mean())


def check_grads(tr, ref_grads, res=None):
    """Gradients of an iteration against the oracle's (DESIGN.md s6 'Tolerances'): relative L2 1e-3 on everything; max
    error 1e-3 of the tensor's maximum on the Gaussians that touch no fragile pixel of `res` (all Gaussians when no `res`
    is given), 5e-3 on the rest -- a flipped skip / exit decision moves one pixel's term of their gradient; per row
    1e-3 relative + the atomic noise floor on >= 99.9 % of the rows.  ref_grads: one dict per partition (None = zeros)."""
    frag = None
    if res is not None:
        H, W = res.image.shape[:2]
        frag = np.zeros(tr.n, bool)
        members = getattr(res, "members", None) or list(range(len(res.proj)))
        for k, m in zip(members, fragile_gaussians(res, W, H)):
            frag[tr.part_offsets[k]:tr.part_offsets[k + 1]] = m
        assert (~frag).any()     # (a fragile pixel has ~50 (near-)contributors; the big footprints of one test scene reach most pixels)
    for key in scenes.PARAM_KEYS:
        w = scenes.PARAM_WIDTH[key]
        got = np32(tr.grads[key]).astype(np.float64).reshape(-1, w)
        ref = np.concatenate([(g[key] if g is not None else np.zeros((tr.part_offsets[k + 1] - tr.part_offsets[k]) * w)).reshape(-1)
                              for k, g in enumerate(ref_grads)]).reshape(-1, w)
        assert rel_l2(got, ref) <= 1e-3, (key, rel_l2(got, ref))
        scale = max(np.abs(ref).max(), 1e-30)
        err = np.abs(got - ref).max(1) / scale
        robust = np.ones(len(err), bool) if frag is None else ~frag
        assert err[robust].max() <= GRAD_MAX_TOL, (key, err[robust].max())
        assert err.max() <= 5e-3, (key, err.max())
        assert grad_rows_close(got, ref, w) >= 0.999, (key, grad_rows_close(got, ref, w))
