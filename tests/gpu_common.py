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
