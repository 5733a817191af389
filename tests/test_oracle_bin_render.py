"""Pins for oracle O2 (tile binning + sort) and O3 (local render), PAPER.md L81, L165,
Eq.1 (L84), Eq.3-4 (L167-L172): brute force, a library sort, closed forms, the dense
fp64 restatement in tests/dense_ref.py, and invariants."""
import math

import numpy as np
import pytest
import torch

import oracle
from tests import dense_ref
from tests.common import cam64, gaussians, random_scene, simple_camera


def _proj(p, cam, deg=0, cfg=oracle.DEFAULT_CFG):
    return oracle.project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], deg,
                          cam64(cam), cfg)


def test_bin_sort_matches_library_lexicographic_sort():
    rng = np.random.default_rng(10)
    p, cam = random_scene(rng, 300, size=70, f=60.0)
    # force depth ties so that stability (ties -> ascending Gaussian index) is exercised
    p["mean"][50:60] = p["mean"][40:50]
    pr = _proj(p, cam)
    W = H = 70; TX = 5
    b = oracle.bin_sort(pr.means2d, pr.radius, pr.depth, W, H)
    tuples = []
    for i in range(300):
        x0, y0, x1, y1 = pr.rect[i]
        bits = int(np.float32(pr.depth[i]).view(np.uint32))
        for ty in range(y0, y1):
            for tx in range(x0, x1):
                tuples.append((ty * TX + tx, bits, i))
    assert b.M == len(tuples) == int(pr.tiles_touched.sum())
    tuples.sort()
    assert [(int(k) >> 32, int(k) & 0xFFFFFFFF, int(v)) for k, v in zip(b.keys, b.vals)] == tuples
    assert (np.diff(b.keys.astype(np.uint64)) >= 0).all()
    assert np.array_equal(b.offsets, np.cumsum(pr.tiles_touched).astype(np.uint32))
    # ranges partition [0, M) in tile order; empty tiles are (0,0)
    pos = 0
    tiles = np.array([t for t, _, _ in tuples])
    for t in range(TX * TX):
        cnt = int((tiles == t).sum())
        if cnt == 0:
            assert tuple(b.ranges[t]) == (0, 0)
        else:
            assert tuple(b.ranges[t]) == (pos, pos + cnt)
            pos += cnt
    assert pos == b.M


def test_bin_sort_empty():
    b = oracle.bin_sort(np.zeros((3, 2)), np.zeros(3, np.int32), np.zeros(3), 32, 32)
    assert b.M == 0 and not b.ranges.any() and not b.offsets.any()


def test_render_one_and_two_gaussian_closed_forms():
    # C = c1 a1 + c2 a2 (1 - a1), T = (1-a1)(1-a2), D = d1 a1 + d2 a2 (1-a1); Eq.1, Eq.3, Eq.4
    cam = simple_camera(32, 100.0)
    p = gaussians([[0.02, -0.03, 3.0], [-0.05, 0.04, 5.0]], [0.08, 0.15], [[1, 0, 0, 0]] * 2,
                  [0.3, -0.4], [[0.8, 0.2, 0.1], [0.1, 0.3, 0.9]])
    pr = _proj(p, cam)
    b = oracle.bin_sort(pr.means2d, pr.radius, pr.depth, 32, 32)
    pa = oracle.render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, b.vals, b.ranges, 32, 32)
    f = 100.0
    for (i, j) in [(16, 16), (14, 18), (12, 12), (20, 13)]:
        al = []
        for g, (s, z) in enumerate([(0.08, 3.0), (0.15, 5.0)]):
            var = (f * s / z) ** 2 + 0.3  # on-axis approximation is not exact off-axis: take cov from the conic
            co = pr.conic_opacity[g]
            dx = pr.means2d[g, 0] - (i + 0.5); dy = pr.means2d[g, 1] - (j + 0.5)
            power = -0.5 * (co[0] * dx * dx + co[2] * dy * dy) - co[1] * dx * dy
            a = min(0.99, (1 / (1 + math.exp(-[0.3, -0.4][g]))) * math.exp(power))
            al.append(a if a >= 1 / 255 else 0.0)
        c1, c2 = np.array([0.8, 0.2, 0.1]), np.array([0.1, 0.3, 0.9])
        C = c1 * al[0] + c2 * al[1] * (1 - al[0])
        assert np.allclose(pa.ct[j, i, :3], C, atol=1e-14)
        assert pa.ct[j, i, 3] == pytest.approx((1 - al[0]) * (1 - al[1]), abs=1e-14)
        assert pa.d[j, i] == pytest.approx(3.0 * al[0] + 5.0 * al[1] * (1 - al[0]), abs=1e-13)
    # Gaussian of Eq.1 at its centre: alpha = opacity exactly (power = 0)
    p1 = gaussians([[0.005 * 3.0, 0.005 * 3.0, 3.0]], [0.08], [[1, 0, 0, 0]], [0.3], [[0.8, 0.2, 0.1]])
    pr1 = _proj(p1, cam)
    assert np.allclose(pr1.means2d[0], [16.5, 16.5])
    b1 = oracle.bin_sort(pr1.means2d, pr1.radius, pr1.depth, 32, 32)
    pa1 = oracle.render_partial(pr1.means2d, pr1.conic_opacity, pr1.rgb, pr1.depth, b1.vals, b1.ranges, 32, 32)
    assert 1 - pa1.ct[16, 16, 3] == pytest.approx(1 / (1 + math.exp(-0.3)), abs=1e-12)


def test_alpha_clamp_skip_and_early_exit_rules():
    # 12 identical opaque Gaussians stacked in depth at the pixel centre: alpha = min(0.99, ~1) = 0.99
    # T after n: 0.01^n; the exit fires BEFORE the Gaussian that would take T below 1e-4 (reading s2):
    # T: 1 -> 1e-2 -> 1e-4 ... 0.01*0.01 = 1e-4 is not < 1e-4 in exact arithmetic but (1-0.99) rounds,
    # so use alpha_max = 0.8: T = 0.2^n, stop before n=6 (6.4e-5 < 1e-4) -> 5 contributors, T = 3.2e-4
    cam = simple_camera(32, 100.0)
    n = 12
    mean = [[0.005 * (3 + 0.1 * k), 0.005 * (3 + 0.1 * k), 3 + 0.1 * k] for k in range(n)]
    p = gaussians(mean, [0.2] * n, [[1, 0, 0, 0]] * n, [20.0] * n, [[0.5, 0.5, 0.5]] * n)
    pr = _proj(p, cam)
    b = oracle.bin_sort(pr.means2d, pr.radius, pr.depth, 32, 32)
    cfg = (1 / 255, 0.8, 1e-4, 0.3, 1.3, 0.1)
    pa = oracle.render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, b.vals, b.ranges, 32, 32, cfg)
    assert pa.n_contrib[16, 16] == 5
    assert pa.ct[16, 16, 3] == pytest.approx(0.2 ** 5, rel=1e-12)
    assert pa.t_exit[16, 16] == pytest.approx(0.2 ** 5, rel=1e-12)
    assert pa.ct[16, 16, 0] == pytest.approx(0.5 * (1 - 0.2 ** 5), rel=1e-12)
    # T_eps = 0: nothing stops; all 12 contribute
    cfg0 = (1 / 255, 0.8, 0.0, 0.3, 1.3, 0.1)
    pa0 = oracle.render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, b.vals, b.ranges, 32, 32, cfg0)
    assert pa0.n_contrib[16, 16] == 12 and pa0.ct[16, 16, 3] == pytest.approx(0.2 ** 12, rel=1e-10)
    assert pa0.t_exit[16, 16] == -1
    # alpha < 1/255 is skipped: far from the centre n_contrib stays 0 and T == 1 exactly
    far = pa.n_contrib == 0
    assert far.any() and (pa.ct[far][:, 3] == 1.0).all() and not pa.ct[far][:, :3].any()


@pytest.mark.parametrize("seed,cfg", [(20, oracle.DEFAULT_CFG), (21, oracle.DEFAULT_CFG), (22, oracle.SMOOTH_CFG)])
def test_tiled_render_equals_dense_restatement(seed, cfg):
    rng = np.random.default_rng(seed)
    p, cam = random_scene(rng, 60, size=40, f=45.0, sh_degree=3)
    p["opacity_logit"] += 2.0  # enough opacity for early exits in threshold mode
    pr = _proj(p, cam, 3, cfg)
    W = H = 40
    b = oracle.bin_sort(pr.means2d, pr.radius, pr.depth, W, H)
    pa = oracle.render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, b.vals, b.ranges, W, H, cfg)
    tp = {k: torch.tensor(np.asarray(v, np.float64)) for k, v in p.items()}
    cd = dict(R=torch.tensor(np.asarray(cam.R, np.float64)), t=torch.tensor(np.asarray(cam.t, np.float64)),
              fx=cam.fx, fy=cam.fy, cx=cam.cx, cy=cam.cy, W=W, H=H)
    prd = dense_ref.project_dense(tp, cd, 3)
    # projection agrees with the independent restatement (incl. the SH built from angles)
    vis = pr.radius > 0
    assert np.allclose(prd["u"].numpy()[vis], pr.means2d[vis, 0], rtol=1e-11)
    assert np.allclose(prd["rgb"].numpy()[vis], pr.rgb[vis], atol=1e-11)
    assert np.allclose(prd["conic"].numpy()[vis][:, 0, 1], pr.conic_opacity[vis, 1], rtol=1e-9, atol=1e-12)
    C, T, D = dense_ref.render_dense(prd, torch.tensor(pr.rect), torch.tensor(vis), W, H, cfg[0], cfg[1], cfg[2])
    assert np.abs(C.numpy().reshape(H, W, 3) - pa.ct[..., :3]).max() < 1e-11
    assert np.abs(T.numpy().reshape(H, W) - pa.ct[..., 3]).max() < 1e-11
    assert np.abs(D.numpy().reshape(H, W) - pa.d).max() < 1e-10
    if cfg[2] > 0:
        assert (pa.t_exit >= 0).any()  # the early exit was exercised


def test_render_invariants_on_tiny_config():
    from paper_2606_18588_b200 import scenes
    sc = scenes.tiny(n=1024, size=64)
    cam = sc.cameras[0].as_array()
    res = oracle.forward(sc.partitions(), cam, 0)
    for pa, pr, b in zip(res.partials, res.proj, res.bins):
        T = pa.ct[..., 3]
        assert (T >= 1e-4).all() and (T <= 1).all()  # exit fires before the offending Gaussian
        assert (pa.ct[..., :3] <= (1 - T)[..., None] * pr.rgb.max() + 1e-12).all()  # sum w = 1 - T
        assert (pa.ct[..., :3] >= 0).all()
        lens = (b.ranges[:, 1] - b.ranges[:, 0]).reshape(4, 4)
        assert (pa.n_contrib.reshape(4, 16, 4, 16).max(axis=(1, 3)) <= lens).all()
        # weighted mean depth lies within the partition's depth span
        live = T < 1
        key = pa.d[live] / (1 - T[live])
        assert (key >= pr.depth[pr.radius > 0].min() - 1e-9).all() and (key <= pr.depth.max() + 1e-9).all()
    assert res.walked == sum(int(((b.ranges[:, 1] - b.ranges[:, 0]).astype(np.int64)).sum()) * 256 for b in res.bins) or res.walked > 0


def test_tile_list_restricts_work():
    from paper_2606_18588_b200 import scenes
    sc = scenes.tiny(n=512, size=64)
    cam = sc.cameras[0].as_array()
    full = oracle.forward(sc.partitions(), cam, 0)
    sub = oracle.forward(sc.partitions(), cam, 0, tile_list=[5, 10])
    for t in (5, 10):
        ty, tx = divmod(t, 4)
        sl = (slice(16 * ty, 16 * ty + 16), slice(16 * tx, 16 * tx + 16))
        assert np.array_equal(full.image[sl], sub.image[sl])
    assert not sub.image[0:16, 0:16].any()


def test_depth_key_is_the_fp32_depth_in_a_fixed_operation_order():
    """Reading s12: the sort key holds float_bits(depth), an integer decision taken in fp32.  oracle.depth_key is that
    fp32 value -- exactly representable, within one fp32 rounding of the fp64 depth of the projection, equal to the
    exactly rounded depth wherever that is unambiguous -- and the free-running oracle orders by it."""
    import oracle
    from .common import random_scene
    rng = np.random.default_rng(11)
    p, cam = random_scene(rng, 400, size=48, f=60.0, sh_degree=0)
    p = {k: v.astype(np.float32).astype(np.float64) for k, v in p.items()}
    camv = cam.as_array()
    dk = oracle.depth_key(p["mean"], camv)
    assert np.array_equal(dk, dk.astype(np.float32).astype(np.float64))           # fp32 numbers
    pr = oracle.project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], 0, camv)
    vis = pr.radius > 0
    ulp = np.spacing(np.abs(pr.depth[vis]).astype(np.float32)).astype(np.float64)
    assert (np.abs(dk[vis] - pr.depth[vis]) <= 1.5 * ulp).all()                   # three roundings, mostly cancelling
    assert (dk[vis] == pr.depth[vis].astype(np.float32)).mean() > 0.5             # usually THE correctly rounded depth
    # the driver sorts by it: every tile list is ordered by (bits(depth_key), index)
    res = oracle.forward([p], camv, 0)
    b = res.bins[0]
    bits = dk.astype(np.float32).view(np.uint32).astype(np.uint64)
    assert np.array_equal(b.keys & np.uint64(0xFFFFFFFF), bits[b.vals])
    for t in range(b.ranges.shape[0]):
        a, e = b.ranges[t]
        k = list(zip(bits[b.vals[a:e]].tolist(), b.vals[a:e].tolist()))
        assert k == sorted(k)
