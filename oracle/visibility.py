"""Oracle for the two optional subsystems -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Visibility prediction and conflict-free view consolidation
(PAPER.md L247-L249), stated as plainly as possible in numpy/scipy on top of the stage oracle
(``oracle/__init__.py``).  Shares no code with the CUDA path.

* ``visible_regions``  L212/L227: partition k is geometrically visible on tile t iff some point of
  its axis-aligned box lies in front of the near plane and projects into the tile's pixel-area
  rectangle.  That definition is written out as one linear feasibility problem per (box, tile)
  and handed to a library LP solver (scipy ``linprog``/HiGHS): no clipping, no hulls.
* ``saturation``       L213/L231: "once the cumulative transmittance prod_{k<=m} T^k is less than a
  threshold eps, all subsequent partitions behind GPU m ... become invisible on the camera ray".
  Per pixel the front product of every partition follows from the composition order of Eq.5;
  a (partition, tile) slot is saturated iff EVERY pixel of the tile is (tile-level reading of the
  per-pixel rule: DESIGN.md s27).
* ``schedule_views``   L249: greedy bucketing in view order.
* ``iteration_plan``   the whole iteration under a plan: B views, each partition rendering at most
  one of them, tile lists of skipped slots dropped, gradients of the views added.
"""
from __future__ import annotations

import numpy as np

from . import (DEFAULT_CFG, TILE, IterationResult, bin_sort, cam_wh, compose, compose_bwd, depth_key, l1, project,
               project_bwd, raster_bwd, render_partial, tiles_xy)

TILE_INVISIBLE, TILE_SATURATED = 1, 2


def _tile_rect(t, TX, W, H):
    tx, ty = t % TX, t // TX
    return 16.0 * tx, min(16.0 * (tx + 1), float(W)), 16.0 * ty, min(16.0 * (ty + 1), float(H))


def _reach(cam, s_max, cfg):
    """Reading s21.  Gaussians belong to a partition by their mean (L155) but their footprints stick out of
    its box (L474); the binning keeps every Gaussian whose square of tiles meets the image.  For scale <= s_max and
    camera-space mean (x, y, z), z > near:  radius = ceil(3 sqrt(lambda)), lambda = mid + sqrt(max(floor, mid^2 - det))
    <= lambda_max(Sigma2D) + sqrt(floor);  Sigma2D = J W Sigma W^T J^T + dilation I  =>  lambda_max <= |J|_2^2 s^2 +
    dilation;  with J = [[fx/z, 0, -fx Lx/z], [0, fy/z, -fy Ly/z]], |Lx| <= limx, |Ly| <= limy (the clamps of s9),
    |J|_2^2 <= c^2/z^2, c^2 = max(fx, fy)^2 (1 + limx^2 + limy^2).  So radius <= 3 c s/z + 3 sqrt(e) + 1,
    e = dilation + sqrt(floor), and the square (pixel columns within radius + 1.5 of u = fx x/z + cx) can meet [0, W]
    only if  -(cx + g) z - h <= fx x <= (W - cx + g) z + h  with g = 2.5 + 3 sqrt(e), h = 3 c s -- linear in the mean;
    likewise in y.  Returns (rows, rhs) of those four half spaces as A p_world <= b, and (c^2, e)."""
    R, t = cam[0:9].reshape(3, 3), cam[9:12]
    fx, fy, cx, cy = cam[12:16]
    W, H = cam_wh(cam)
    dilation, lim_factor, rfloor = cfg[3], cfg[4], cfg[5]
    limx, limy = lim_factor * W / (2 * fx), lim_factor * H / (2 * fy)
    c2 = max(fx, fy) ** 2 * (1 + limx * limx + limy * limy)
    e = dilation + np.sqrt(rfloor)
    g, h = 2.5 + 3 * np.sqrt(e), 3 * np.sqrt(c2) * s_max
    rows, rhs = [], []
    # fx xc - (W - cx + g) zc <= h   with xc = R0.p + t0, zc = R2.p + t2
    for sign, f, axis, span in ((1.0, fx, 0, W - cx), (-1.0, fx, 0, cx), (1.0, fy, 1, H - cy), (-1.0, fy, 1, cy)):
        a = sign * f * R[axis] - (span + g) * R[2]
        rows.append(a); rhs.append(h - (sign * f * t[axis] - (span + g) * t[2]))
    return rows, rhs, c2, e


def visible_regions(aabb_lo, aabb_hi, cam, tiles=None, tol=1e-7, max_scale=None, cfg=DEFAULT_CFG, whole_image=False):
    """state[n_boxes, tiles] (0 = visible, TILE_INVISIBLE, 255 = tile not evaluated), participants bitmask (one bit per
    box), margin[n_boxes, tiles] = the largest slack s for which  A p + s <= b  is still feasible inside the box
    (rows scaled to unit norm; > 0 robustly visible, < 0 robustly invisible, |s| <= tol undecided).
    max_scale None: the plain region of L212 (box ^ {z >= near} projected).  max_scale[n_boxes] (boxes of MEANS, the
    largest scale of their Gaussians): the conservative region of reading s21 -- the box is first cut down to the
    means that can reach the image (`_reach`), z_min of what is left gives the margin m = 3 sqrt(c^2 s^2/z_min^2 + e)
    + 3.5 px by which every tile rectangle is grown.  whole_image: one 'tile' = the image rectangle (participants only)."""
    from scipy.optimize import linprog
    cam = np.asarray(cam, np.float64)
    R, t = cam[0:9].reshape(3, 3), cam[9:12]
    fx, fy, cx, cy = cam[12:16]
    W, H = cam_wh(cam)
    near = cam[18]
    TX, TY = tiles_xy(W, H)
    lo = np.asarray(aabb_lo, np.float64).reshape(-1, 3)
    hi = np.asarray(aabb_hi, np.float64).reshape(-1, 3)
    K = lo.shape[0]
    if whole_image:
        tiles = [0]
    else:
        tiles = range(TX * TY) if tiles is None else [int(x) for x in tiles]
    state = np.full((K, 1 if whole_image else TX * TY), 255, np.uint8)
    margin = np.full(state.shape, np.nan)
    part = 0
    for k in range(K):
        bounds = [(lo[k, 0], hi[k, 0]), (lo[k, 1], hi[k, 1]), (lo[k, 2], hi[k, 2])]
        xrows, xrhs, mg = [], [], 0.0
        if max_scale is not None:
            xrows, xrhs, c2, e = _reach(cam, float(max_scale[k]), cfg)
            # z_min over the means that can reach the image (and lie in front of the near plane)
            res = linprog(c=R[2], A_ub=np.array([-R[2]] + xrows), b_ub=np.array([t[2] - near] + xrhs), bounds=bounds, method="highs")
            if res.status != 0:                     # no mean of this box can reach the image
                state[k, list(tiles)] = TILE_INVISIBLE
                margin[k, list(tiles)] = -1.0
                continue
            zmin = max(near, float(R[2] @ res.x + t[2]))
            mg = 3.0 * np.sqrt(c2 * float(max_scale[k]) ** 2 / zmin ** 2 + e) + 3.5
        for tl in tiles:
            x0, x1, y0, y1 = (0.0, float(W), 0.0, float(H)) if whole_image else _tile_rect(tl, TX, W, H)
            x0, x1, y0, y1 = x0 - mg, x1 + mg, y0 - mg, y1 + mg
            # camera-space coordinates are affine in the world point p: xc = R0.p + t0 etc.
            rows, rhs = [], []
            rows.append(-R[2]); rhs.append(t[2] - near)                                   # zc >= near
            rows.append(-(fx * R[0] + (cx - x0) * R[2])); rhs.append(fx * t[0] + (cx - x0) * t[2])   # u >= x0
            rows.append(fx * R[0] + (cx - x1) * R[2]); rhs.append(-(fx * t[0] + (cx - x1) * t[2]))   # u <= x1
            rows.append(-(fy * R[1] + (cy - y0) * R[2])); rhs.append(fy * t[1] + (cy - y0) * t[2])   # v >= y0
            rows.append(fy * R[1] + (cy - y1) * R[2]); rhs.append(-(fy * t[1] + (cy - y1) * t[2]))   # v <= y1
            A = np.array(rows + xrows); b = np.array(rhs + xrhs)
            nrm = np.linalg.norm(A, axis=1)
            A = A / nrm[:, None]; b = b / nrm
            # maximise s subject to A p + s <= b, lo <= p <= hi
            res = linprog(c=[0, 0, 0, -1.0], A_ub=np.hstack([A, np.ones((len(b), 1))]), b_ub=b,
                          bounds=bounds + [(None, 1e6)], method="highs")
            assert res.status == 0, res.message
            s = float(res.x[3])
            margin[k, tl] = s
            state[k, tl] = 0 if s >= 0 else TILE_INVISIBLE
            if s >= 0:
                part |= 1 << k
    return state, part, margin


def participants(aabb_lo, aabb_hi, cam, max_scale=None, cfg=DEFAULT_CFG):
    """GetParticipants(v) (L249) without the tile grid: `visible_regions` posed for the whole image at once (one bit
    per box)."""
    return visible_regions(aabb_lo, aabb_hi, cam, max_scale=max_scale, cfg=cfg, whole_image=True)[1]


def union_regions(state_boxes, box_part, K):
    """A partition covered by several boxes is visible on a tile iff one of its boxes is (state per box -> per partition)."""
    state_boxes = np.asarray(state_boxes)
    out = np.full((K, state_boxes.shape[1]), TILE_INVISIBLE, np.uint8)
    for j, k in enumerate(box_part):
        out[k][state_boxes[j] == 0] = 0
    return out


def ray_hits_box(aabb_lo, aabb_hi, cam, u, v):
    """Brute-force pin for ``visible_regions``: does the camera ray through image point (u, v) meet the box
    at camera depth >= near?  (slab test along the ray, parameterised by the camera depth z)."""
    cam = np.asarray(cam, np.float64)
    R, t = cam[0:9].reshape(3, 3), cam[9:12]
    fx, fy, cx, cy = cam[12:16]
    near = cam[18]
    dcam = np.array([(u - cx) / fx, (v - cy) / fy, 1.0])    # point at depth z is z * dcam in camera space
    o = -R.T @ t
    dw = R.T @ dcam                                          # world point = o + z * dw
    zlo, zhi = near, np.inf
    for a in range(3):
        if abs(dw[a]) < 1e-300:
            if not (aabb_lo[a] <= o[a] <= aabb_hi[a]):
                return False
            continue
        z0, z1 = (aabb_lo[a] - o[a]) / dw[a], (aabb_hi[a] - o[a]) / dw[a]
        zlo, zhi = max(zlo, min(z0, z1)), min(zhi, max(z0, z1))
    return zlo <= zhi


def apply_tile_state(ranges, state_k):
    """a skipped (partition, tile) slot loses its list (range = (0,0)); keys are untouched."""
    r = np.array(ranges, copy=True).reshape(-1, 2)
    r[np.asarray(state_k).reshape(-1) != 0] = 0
    return r


def front_products(ct, order):
    """front[k,H,W] = product of the T^j composited in front of partition k at each pixel, from the
    composition order of Eq.5 (order[H,W,K], front first)."""
    K, H, W, _ = ct.shape
    T = np.moveaxis(np.asarray(ct)[..., 3], 0, -1)                         # [H,W,K]
    Tord = np.take_along_axis(T, order.astype(np.int64), axis=-1)          # T in composition order
    excl = np.concatenate([np.ones((H, W, 1)), np.cumprod(Tord, axis=-1)[..., :-1]], axis=-1)
    front = np.empty((H, W, K))
    np.put_along_axis(front, order.astype(np.int64), excl, axis=-1)
    return np.moveaxis(front, -1, 0)


def saturation(ct, d, eps, state_in=None, members=None):
    """Returns (state_out[K,tiles], margin[K,tiles]).  state_out = (state_in & INVISIBLE) | SATURATED iff the
    front product of partition k is < eps at EVERY pixel of the tile; margin = min over the tile's pixels of
    |front - eps| / eps (a slot whose decision hinges on a pixel within fp32 rounding of eps is fragile).
    members: partitions composed together (default all K); others are left at state_in."""
    ct = np.asarray(ct, np.float64); d = np.asarray(d, np.float64)
    K, H, W, _ = ct.shape
    TX, TY = tiles_xy(W, H)
    members = list(range(K)) if members is None else list(members)
    _, _, order, _ = compose(ct[members], d[members])
    front = front_products(ct[members], order)                            # [len(members),H,W]
    out = np.zeros((K, TX * TY), np.uint8) if state_in is None else np.array(state_in, np.uint8).reshape(K, -1).copy()
    margin = np.full((K, TX * TY), np.inf)
    for j, k in enumerate(members):
        for tl in range(TX * TY):
            x0, x1, y0, y1 = (int(a) for a in _tile_rect(tl, TX, W, H))
            f = front[j, y0:y1, x0:x1]
            sat = bool(np.all(f < eps))
            out[k, tl] = (out[k, tl] & TILE_INVISIBLE) | (TILE_SATURATED if sat else 0)
            margin[k, tl] = float(np.min(np.abs(f - eps))) / eps if eps > 0 else np.inf
    return out, margin


def schedule_views(participants, max_views_per_bucket=8):
    """L249: "iterate over all camera views to greedily and incrementally bucket more views that have no
    overlap with the GPUs in the existing buckets ... If no compatible bucket is found, a new bucket is created"."""
    used, count, out = [], [], []
    for p in participants:
        for j in range(len(used)):
            if used[j] & p == 0 and count[j] < max_views_per_bucket:
                break
        else:
            used.append(0); count.append(0); j = len(used) - 1
        used[j] |= p; count[j] += 1
        out.append(j)
    return out, len(used)


def iteration_plan(parts, cams, view_of_part, sh_degree, targets, bg=(0.0, 0.0, 0.0), cfg=DEFAULT_CFG,
                   tile_state=None, g_images=None):
    """One iteration under a plan.  parts: K dicts; cams: B camera arrays (same size); view_of_part[k] in
    {-1, 0..B-1}; tile_state[K,tiles] or None; targets[B] (mean-L1 per view) or g_images[B] given directly.
    Returns a list of B IterationResult (lists indexed by the view's own partitions, .members = their k) and
    grads[K] (dict per partition, zeros for non-participants)."""
    K, B = len(parts), len(cams)
    W, H = cam_wh(cams[0])
    views = []
    grads = [None] * K
    for b in range(B):
        cam = cams[b]
        members = [k for k in range(K) if view_of_part[k] == b]
        res = IterationResult()
        res.members = members
        for k in members:
            p = parts[k]
            pr = project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], sh_degree, cam, cfg)
            bn = bin_sort(pr.means2d, pr.radius, depth_key(p["mean"], cam), W, H)     # order by the fp32 key (s12)
            if tile_state is not None:
                bn.ranges = apply_tile_state(bn.ranges, tile_state[k])
            pa = render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, bn.vals, bn.ranges, W, H, cfg)
            res.proj.append(pr); res.bins.append(bn); res.partials.append(pa)
        if members:
            ct = np.stack([pa.ct for pa in res.partials]); d = np.stack([pa.d for pa in res.partials])
        else:
            ct = np.zeros((0, H, W, 4)); d = np.zeros((0, H, W))
        if members:
            res.image, res.T_total, res.order, res.order_margin = compose(ct, d, bg)
        else:
            res.image = np.broadcast_to(np.asarray(bg, np.float64), (H, W, 3)).copy(); res.T_total = np.ones((H, W))
        if g_images is not None:
            g_image = np.asarray(g_images[b], np.float64)
        else:
            res.loss, g_image = l1(res.image, targets[b])
        res.g_image = g_image
        if members:
            res.g_ct = compose_bwd(ct, d, g_image, bg)
        for j, k in enumerate(members):
            p, pr, bn = parts[k], res.proj[j], res.bins[j]
            g2 = raster_bwd(pr.means2d, pr.conic_opacity, pr.rgb, bn.vals, bn.ranges, W, H, res.g_ct[j], cfg)
            grads[k] = project_bwd(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], sh_degree, cam,
                                   pr.radius, pr.clamp, *g2, cfg=cfg)
            res.grads2d.append(g2)
        views.append(res)
    for k in range(K):
        if grads[k] is None:
            n = int(np.asarray(parts[k]["opacity_logit"]).shape[0])
            grads[k] = dict(mean=np.zeros((n, 3)), log_scale=np.zeros((n, 3)), quat=np.zeros((n, 4)),
                            opacity_logit=np.zeros(n), sh=np.zeros((n, 16, 3)))
    return views, grads


def adam_rows(param, grad, m, v, rows, lr, beta1=0.9, beta2=0.999, eps=1e-15, step=1):
    """Visible-only Adam (an option OUTSIDE the paper, SURVEY.md s8(f) NEXT 4 / DESIGN.md s31): the Adam step of
    ``oracle.adam`` on the boolean-selected ``rows`` of [n, w] float64 arrays, in place; the other rows keep their
    parameters and both moments (no decay).  The bias correction uses the global ``step``."""
    from . import adam
    rows = np.asarray(rows, bool)
    p = np.ascontiguousarray(param[rows]); mm = np.ascontiguousarray(m[rows]); vv = np.ascontiguousarray(v[rows])
    adam(p.reshape(-1), np.ascontiguousarray(grad[rows]).reshape(-1), mm.reshape(-1), vv.reshape(-1), lr, beta1, beta2, eps, step)
    param[rows] = p; m[rows] = mm; v[rows] = vv
