"""Pins of the oracle for the two optional subsystems (oracle/visibility.py) and of the product's HOST logic
(splx_visible_regions, splx_schedule_views need no GPU): PAPER.md L212-L231 (visibility prediction),
L247-L249 (conflict-free consolidation)."""
import numpy as np
import pytest

import oracle
from oracle import visibility as ov
from paper_2606_18588_b200 import binding, scenes

from .common import cam64, random_scene


def _cam(width=96, height=80, pitch=40.0, yaw=30.0, alt=30.0, target=(1.3, -0.7, 0.0)):
    return scenes.aerial_camera(width, height, 60.0, alt, pitch, yaw, target)


BOXES_LO = np.array([[-20, -20, 0], [0, -20, 0], [-20, 0, 0], [0, 0, 0], [200, 200, 0], [-3, -3, 0]], np.float32)
BOXES_HI = np.array([[0, 0, 8], [20, 0, 8], [0, 20, 8], [20, 20, 8], [220, 220, 8], [3, 3, 0]], np.float32)


def test_region_lp_agrees_with_ray_brute_force():
    """The LP statement against geometry done the slow way: every sampled image point whose ray meets the
    box lies in a visible tile, and a robustly visible tile contains a point whose ray meets the box."""
    cam = _cam()
    c64 = cam.as_array()
    state, part, margin = ov.visible_regions(BOXES_LO, BOXES_HI, c64)
    W, H = cam.width, cam.height
    TX = (W + 15) // 16
    us = np.arange(0.125, W, 0.25); vs = np.arange(0.125, H, 0.25)
    for k in range(len(BOXES_LO)):
        hit_tiles = set()
        for v in vs:
            for u in us:
                if ov.ray_hits_box(BOXES_LO[k].astype(np.float64), BOXES_HI[k].astype(np.float64), c64, u, v):
                    hit_tiles.add(int(v // 16) * TX + int(u // 16))
        vis_tiles = set(np.nonzero(state[k] == 0)[0].tolist())
        assert hit_tiles <= vis_tiles, k
        for t in vis_tiles - hit_tiles:          # only slivers thinner than the sampling pitch may be missed
            assert margin[k, t] < 0.2, (k, t, margin[k, t])
    assert part & 0b1111 == 0b1111 and not (part >> 4) & 1   # the four central boxes are seen, the far one is not


def test_region_of_a_box_that_fills_the_view_or_lies_behind_the_camera():
    cam = _cam()
    c64 = cam.as_array()
    state, part, _ = ov.visible_regions(np.array([[-500, -500, -5]], np.float32), np.array([[500, 500, 5]], np.float32), c64)
    assert part == 1 and np.all(state == 0)                   # the ground slab covers every tile
    o = -cam.R.T.astype(np.float64) @ cam.t.astype(np.float64)
    fwd = cam.R[2].astype(np.float64)
    behind = o - 50.0 * fwd
    state, part, _ = ov.visible_regions((behind - 1).astype(np.float32)[None], (behind + 1).astype(np.float32)[None], c64)
    assert part == 0 and np.all(state == ov.TILE_INVISIBLE)


def test_library_host_geometry_equals_the_lp_oracle():
    """splx_visible_regions (clip + hull + separating axes, host C++) against the LP, on every tile whose
    LP margin is not within rounding of zero."""
    for yaw, pitch in ((30.0, 40.0), (200.0, 25.0), (95.0, 70.0)):
        cam = _cam(yaw=yaw, pitch=pitch)
        ref, part_ref, margin = ov.visible_regions(BOXES_LO, BOXES_HI, cam.as_array())
        got, part = binding.visible_regions(BOXES_LO, BOXES_HI, cam)
        robust = np.abs(margin) > 1e-6
        assert robust.mean() > 0.98
        assert np.array_equal(got[robust], ref[robust])
        assert part == part_ref


def test_participants_is_the_union_of_the_tile_regions():
    """ov.participants (one LP per box over the whole image) == 'some tile of visible_regions is visible', for the plain
    and for the conservative regions, and == the library's host geometry."""
    for yaw, pitch in ((30.0, 40.0), (200.0, 25.0)):
        cam = _cam(yaw=yaw, pitch=pitch)
        c64 = cam.as_array()
        for ms in (None, np.array([0.0, 0.1, 0.5, 2.0, 30.0, 0.2])):
            state, part_ref, _ = ov.visible_regions(BOXES_LO, BOXES_HI, c64, max_scale=ms)
            assert ov.participants(BOXES_LO, BOXES_HI, c64, ms) == part_ref
            assert binding.visible_regions(BOXES_LO, BOXES_HI, cam, ms)[1] == part_ref


def test_schedule_views_is_greedy_and_conflict_free():
    rng = np.random.default_rng(3)
    for trial in range(20):
        n = int(rng.integers(1, 30))
        parts = [int(rng.integers(1, 1 << 8)) & int(rng.integers(1, 1 << 8)) or 1 for _ in range(n)]
        cap = int(rng.integers(1, 9))
        ref, nb_ref = ov.schedule_views(parts, cap)
        got, nb = binding.schedule_views(parts, cap)
        assert got == ref and nb == nb_ref
        for b in range(nb):
            members = [parts[i] for i in range(n) if got[i] == b]
            assert 1 <= len(members) <= cap
            acc = 0
            for m in members:
                assert acc & m == 0
                acc |= m
    # Fig. 15 of the paper: V0 needs GPUs {0,2}, V2 needs {1,3}: one slot; a view on {0,1} conflicts with both
    assert ov.schedule_views([0b0101, 0b0011, 0b1010])[0] == [0, 1, 0]


def _two_layer_partials(H=32, W=32):
    """K = 3 hand-made partials: partition 0 in front (D/(1-T) = 1), 1 behind it (2), 2 empty."""
    ct = np.zeros((3, H, W, 4)); d = np.zeros((3, H, W))
    ct[..., 3] = 1.0
    ct[0, ..., :3] = 0.3; ct[0, ..., 3] = 5e-5; d[0] = 1.0 * (1 - 5e-5)
    ct[1, ..., :3] = 0.2; ct[1, ..., 3] = 0.5; d[1] = 2.0 * 0.5
    return ct, d


def test_saturation_closed_forms():
    ct, d = _two_layer_partials()
    ct[0, 0:16, 0:16, 3] = 0.5; d[0, 0:16, 0:16] = 0.5          # tile 0: front partition is half transparent
    ct[0, 20, 20, 3] = 0.9; d[0, 20, 20] = 0.1                   # tile 3: one unsaturated pixel
    state, margin = ov.saturation(ct, d, 1e-4)
    # partition 0 is in front everywhere: never saturated.  1 is behind T = 5e-5 < eps except tile 0 and the
    # pixel in tile 3.  2 (empty) stands behind both: 5e-5 * 0.5 < eps except tile 0 (0.25) and that pixel.
    assert state[0].tolist() == [0, 0, 0, 0]
    assert state[1].tolist() == [0, 2, 2, 0]
    assert state[2].tolist() == [0, 2, 2, 0]
    # geometric bit is preserved, saturated bit recomputed
    s_in = np.array([[1, 0, 0, 0], [0, 0, 2, 2], [1, 1, 0, 0]], np.uint8)
    state2, _ = ov.saturation(ct, d, 1e-4, s_in)
    assert state2.tolist() == [[1, 0, 0, 0], [0, 2, 2, 0], [1, 3, 2, 0]]
    # a larger threshold saturates more (Table 4 sweeps eps): with eps = 0.3, 0.25 < eps on tile 0 for partition 2
    state3, _ = ov.saturation(ct, d, 0.3)
    assert state3[2].tolist() == [2, 2, 2, 0] and state3[1, 0] == 0


def test_skipping_saturated_tiles_changes_the_image_by_at_most_eps():
    """every skipped slot has front product < eps, so dropping it moves a pixel by <= eps * max rgb."""
    sc = scenes.small_city(n=6000, width=96, height=80, n_views=1)
    cam = sc.cameras[0].as_array()
    parts = sc.partitions()
    eps = 1e-2
    views, _ = ov.iteration_plan(parts, [cam], [0] * sc.K, sc.sh_degree, sc.targets)
    res = views[0]
    ct = np.stack([p.ct for p in res.partials]); d = np.stack([p.d for p in res.partials])
    state, _ = ov.saturation(ct, d, eps)
    front = ov.front_products(ct, res.order)
    TX = (sc.cameras[0].width + 15) // 16
    n_skipped = 0
    for k in range(sc.K):
        for t in np.nonzero(state[k])[0]:
            x0, y0 = (t % TX) * 16, (t // TX) * 16
            assert np.all(front[k, y0:y0 + 16, x0:x0 + 16] < eps)
            n_skipped += int(res.bins[k].ranges.reshape(-1, 2)[t, 1] > res.bins[k].ranges.reshape(-1, 2)[t, 0])
    views2, _ = ov.iteration_plan(parts, [cam], [0] * sc.K, sc.sh_degree, sc.targets, tile_state=state)
    rgb_max = max(float(p.rgb.max()) for p in res.proj)
    assert np.abs(views2[0].image - res.image).max() <= eps * rgb_max * (1 + 1e-9)
    assert n_skipped > 0, "the test scene must saturate somewhere"


def test_plan_with_one_view_is_the_plain_iteration():
    rng = np.random.default_rng(5)
    p, cam = random_scene(rng, 60, size=48, f=60.0)
    parts = [{k: v[:30] for k, v in p.items()}, {k: v[30:] for k, v in p.items()}]
    target = rng.uniform(0, 1, (48, 48, 3))
    ref = oracle.iteration(parts, cam64(cam), 3, target)
    views, grads = ov.iteration_plan(parts, [cam64(cam)], [0, 0], 3, [target])
    assert np.array_equal(views[0].image, ref.image)
    for k in range(2):
        for key in oracle.PARAM_KEYS:
            assert np.array_equal(grads[k][key], ref.grads[k][key])


def test_consolidated_views_equal_the_views_one_by_one():
    """L249: views of a conflict-free bucket touch disjoint partitions, so one consolidated pass = the two
    single-view passes over their own partitions; a non-participant gets no gradient."""
    rng = np.random.default_rng(6)
    p, cam_a = random_scene(rng, 90, size=48, f=60.0)
    cam_b = scenes.Camera(cam_a.R, cam_a.t + np.array([0.3, -0.2, 0.5]), 55.0, 55.0, 24.0, 24.0, 48, 48)
    parts = [{k: v[i:i + 30] for k, v in p.items()} for i in (0, 30, 60)]
    ta, tb = rng.uniform(0, 1, (48, 48, 3)), rng.uniform(0, 1, (48, 48, 3))
    views, grads = ov.iteration_plan(parts, [cam64(cam_a), cam64(cam_b)], [1, -1, 0], 3, [ta, tb])
    ra = oracle.iteration([parts[2]], cam64(cam_a), 3, ta)
    rb = oracle.iteration([parts[0]], cam64(cam_b), 3, tb)
    assert np.array_equal(views[0].image, ra.image) and np.array_equal(views[1].image, rb.image)
    for key in oracle.PARAM_KEYS:
        assert np.array_equal(grads[2][key], ra.grads[0][key])
        assert np.array_equal(grads[0][key], rb.grads[0][key])
        assert not grads[1][key].any()


def test_kd_partition_is_balanced_and_axis_aligned():
    """median splits along the widest axis: counts differ by at most one per level, the cells are
    disjoint axis-aligned boxes, the imbalance ratio N_max / N_mean - 1 is ~0; a skewed cloud stays balanced where
    a uniform grid does not."""
    rng = np.random.default_rng(8)
    pts = np.concatenate([rng.normal(0, 1, (7001, 3)) * (5, 1, 0.2), rng.normal((30, 4, 0), 0.5, (3000, 3))]).astype(np.float32)
    for K in (1, 2, 8, 16):
        pid = scenes.kd_partition(pts, K)
        counts = np.bincount(pid, minlength=K)
        assert counts.sum() == len(pts) and counts.max() - counts.min() <= 1
        offs = np.concatenate([[0], np.cumsum(counts)])
        assert scenes.imbalance_ratio(offs) <= K / len(pts) + 1e-12       # at most one Gaussian above the mean
        lo = np.array([pts[pid == k].min(0) for k in range(K)]); hi = np.array([pts[pid == k].max(0) for k in range(K)])
        for a in range(K):
            for b in range(a + 1, K):      # boxes of two leaves are separated along some axis (touching at most)
                assert np.any(lo[a] >= hi[b]) or np.any(lo[b] >= hi[a]), (K, a, b)
    first = scenes.kd_partition(pts, 2)
    ext = pts.max(0) - pts.min(0)
    axis = int(np.argmax(ext))
    assert pts[first == 0][:, axis].max() <= pts[first == 1][:, axis].min()        # split along the widest axis
    gid = scenes.grid_partition(pts, pts.min(0)[:2], pts.max(0)[:2], 4, 2)
    g_offs = np.concatenate([[0], np.cumsum(np.bincount(gid, minlength=8))])
    assert scenes.imbalance_ratio(g_offs) > 1.0
    sc = scenes.aerial(n=5000, width=64, height=48, grid=(2, 2), partition="kd", name="kd")
    assert np.diff(sc.part_offsets).tolist() == [1250, 1250, 1250, 1250]


def test_adam_rows_is_adam_on_the_selected_rows():
    """The visible-only option: all rows selected = dense Adam; no row selected = nothing moves; a partial selection
    moves exactly the selected rows, with torch.optim.Adam's values on them (bias correction by the global step)."""
    import torch
    rng = np.random.default_rng(12)
    p0 = rng.standard_normal((50, 3)); g = rng.standard_normal((50, 3))
    rows = rng.uniform(size=50) < 0.4
    p = p0.copy(); m = np.zeros_like(p); v = np.zeros_like(p)
    ov.adam_rows(p, g, m, v, np.zeros(50, bool), 1e-2)
    assert np.array_equal(p, p0) and not m.any() and not v.any()
    pa = p0.copy(); ma = np.zeros_like(p); va = np.zeros_like(p)
    ov.adam_rows(pa, g, ma, va, np.ones(50, bool), 1e-2)
    pd = p0.copy().reshape(-1); md = np.zeros(150); vd = np.zeros(150)
    oracle.adam(pd, g.reshape(-1), md, vd, 1e-2)
    assert np.array_equal(pa.reshape(-1), pd)
    ov.adam_rows(p, g, m, v, rows, 1e-2, step=1)
    t = torch.tensor(p0[rows], dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([t], lr=1e-2, eps=1e-15)
    t.grad = torch.tensor(g[rows]); opt.step()
    assert np.allclose(p[rows], t.detach().numpy(), rtol=1e-12, atol=1e-14)
    assert np.array_equal(p[~rows], p0[~rows]) and not m[~rows].any()


def _margin_scene(seed, n=1500):
    """Gaussians in a 24 x 24 x 6 m slab cut into 2 x 2 cells, scales up to ~1.5 m, seen by a low oblique camera:
    big footprints, many of them cut by the image border."""
    rng = np.random.default_rng(seed)
    mean = np.stack([rng.uniform(-12, 12, n), rng.uniform(-12, 12, n), rng.uniform(0, 6, n)], 1).astype(np.float32)
    p = dict(mean=mean, log_scale=rng.normal(-1.2, 0.7, (n, 3)).astype(np.float32),
             quat=rng.standard_normal((n, 4)).astype(np.float32), opacity_logit=rng.normal(0, 1, n).astype(np.float32),
             sh=np.zeros((n, 16, 3), np.float32))
    pid = scenes.grid_partition(mean, (-12, -12), (12, 12), 2, 2)
    params, offs = scenes._order_by_partition(p, pid, 4)
    cam = scenes.aerial_camera(160, 96, 70.0, 9.0, 28.0, 35.0 + 90 * seed, (2.0, -1.0, 0.0))
    return params, offs, cam


def test_footprint_radius_bound_of_reading_s21():
    """The inequality the conservative regions rest on, against the projection oracle's own radii, Gaussian by Gaussian:
    radius <= 3 c s / z + 3 sqrt(e) + 1 with c^2 = max(fx, fy)^2 (1 + limx^2 + limy^2), e = dilation + sqrt(floor),
    s the Gaussian's largest scale, z its camera depth -- and it is not loose by more than the clamp factor."""
    worst = 0.0
    for seed in range(3):
        params, offs, cam = _margin_scene(seed)
        c64 = cam.as_array()
        pr = oracle.project(params["mean"], params["log_scale"], params["quat"], params["opacity_logit"], params["sh"], 0, c64)
        vis = pr.radius > 0
        assert vis.sum() > 200
        dil, limf, rfl = oracle.DEFAULT_CFG[3:6]
        limx, limy = limf * cam.width / (2 * cam.fx), limf * cam.height / (2 * cam.fy)
        c = max(cam.fx, cam.fy) * np.sqrt(1 + limx ** 2 + limy ** 2)
        e = dil + np.sqrt(rfl)
        smax = np.exp(params["log_scale"].astype(np.float64).max(1))
        bound = 3 * c * smax[vis] / pr.depth[vis] + 3 * np.sqrt(e) + 1
        assert (pr.radius[vis] <= bound).all()
        worst = max(worst, float((pr.radius[vis] / bound).max()))
    assert worst > 0.5          # tight within the factor sqrt(1 + limx^2 + limy^2) of the J clamp


def test_conservative_regions_never_drop_a_list():
    """Boxes of means + max_scale (reading s21): a (partition, tile) slot marked invisible has an EMPTY list in the
    oracle's binning, and a non-participant has no visible Gaussian -- for the LP oracle and for the library's host
    geometry alike, with one box per partition and with sub-cells (which mark MORE slots invisible, still without
    cutting a list)."""
    for seed in range(3):
        params, offs, cam = _margin_scene(seed)
        c64 = cam.as_array()
        bins = []
        for k in range(4):
            a, b = int(offs[k]), int(offs[k + 1])
            pr = oracle.project(params["mean"][a:b], params["log_scale"][a:b], params["quat"][a:b],
                                params["opacity_logit"][a:b], params["sh"][a:b], 0, c64)
            bins.append(oracle.bin_sort(pr.means2d, pr.radius, pr.depth, cam.width, cam.height))
        n_inv = {}
        for sub in (1, 3):
            lo, hi, ms, bp = scenes.partition_boxes(params, offs, sub=sub)
            assert set(bp.tolist()) == {0, 1, 2, 3}
            m = params["mean"]
            for j in range(len(bp)):         # max_scale[j] really bounds the Gaussians of box j
                a, b = int(offs[bp[j]]), int(offs[bp[j] + 1])
                inside = ((m[a:b] >= lo[j]) & (m[a:b] <= hi[j])).all(1)
                assert inside.any() and np.exp(params["log_scale"][a:b][inside].max()) <= ms[j]
            got, part = binding.visible_regions(lo, hi, cam, ms, bp, 4)
            per_box, _, slack = ov.visible_regions(lo, hi, c64, max_scale=ms)
            ref = ov.union_regions(per_box, bp, 4)
            # a tile is decided robustly if every box of the partition is decided robustly on it
            robust = np.ones_like(ref, bool)
            for j, k in enumerate(bp):
                robust[k] &= np.abs(slack[j]) > 1e-6
            assert robust.mean() > 0.97
            assert np.array_equal(got[robust], ref[robust])
            assert part == sum(1 << k for k in range(4) if (ref[k] == 0).any())
            for k in range(4):
                live = bins[k].ranges[:, 1] > bins[k].ranges[:, 0]
                for st in (got[k], ref[k]):
                    assert not (live & (st == ov.TILE_INVISIBLE)).any(), (seed, sub, k)
                if not (part >> k) & 1:
                    assert bins[k].M == 0
            n_inv[sub] = int((got == ov.TILE_INVISIBLE).sum())
        assert n_inv[3] >= n_inv[1]
        # ... while the plain boxes of the means (L212 as printed) do cut lists: the reason for the reading
        lo, hi, ms, bp = scenes.partition_boxes(params, offs)
        bare, _ = binding.visible_regions(lo, hi, cam)
        cut = sum(int(((bins[k].ranges[:, 1] > bins[k].ranges[:, 0]) & (bare[k] == ov.TILE_INVISIBLE)).sum()) for k in range(4))
        assert cut > 0


def test_conservative_region_of_a_box_behind_or_beside_the_camera_is_empty():
    """A box that straddles the camera plane far to the side, or lies wholly behind it, cannot reach the image however
    the near plane cuts it: the reach half spaces remove it (without them z_min = near would blow the margin up)."""
    cam = _cam(width=160, height=96, pitch=45.0, alt=200.0, target=(0.0, 0.0, 0.0))
    o = -cam.R.T.astype(np.float64) @ cam.t.astype(np.float64)
    right, fwd = cam.R[0].astype(np.float64), cam.R[2].astype(np.float64)
    centres = [o + 400.0 * right, o - 300.0 * fwd, o + 300.0 * fwd]          # beside (straddling z = 0), behind, in front
    lo = np.array([c - 60.0 for c in centres], np.float32); hi = np.array([c + 60.0 for c in centres], np.float32)
    ms = np.array([3.0, 3.0, 3.0], np.float32)
    got, part = binding.visible_regions(lo, hi, cam, ms)
    _, part_ref, _ = ov.visible_regions(lo, hi, cam.as_array(), max_scale=ms, whole_image=True)
    assert part == part_ref == 0b100
    assert (got[0] == ov.TILE_INVISIBLE).all() and (got[1] == ov.TILE_INVISIBLE).all() and (got[2] == 0).any()
