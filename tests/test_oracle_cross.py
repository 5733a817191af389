"""Pins of oracle/cross_boundary.py (Fig. 25).  The readings of "spatial support" and
D_overlap are DESIGN.md s32 and cannot be pinned to the paper (parity unpinned); what the mathematics and the
paper's worked example fix is pinned here."""
import numpy as np

import oracle
from oracle import cross_boundary as oc
from oracle import visibility as ov

from .common import gaussians, simple_camera


def test_support_box_is_the_bounding_box_of_the_sigma_ellipsoid():
    """Sample the surface {mu + sigma * R S u, |u| = 1} densely: no point leaves the box, and every face is
    reached to within the sampling resolution."""
    rng = np.random.default_rng(5)
    n = 6
    ls = rng.normal(-1.0, 0.7, (n, 3)); q = rng.standard_normal((n, 4)) * rng.uniform(0.3, 3.0, (n, 1))
    h = oc.support_half_extent(ls, q, 3.0)
    u = rng.standard_normal((200000, 3)); u /= np.linalg.norm(u, axis=1, keepdims=True)
    R = oc.rotation(q)
    for i in range(n):
        pts = 3.0 * (u * np.exp(ls[i])) @ R[i].T
        ext = np.abs(pts).max(axis=0)
        assert np.all(ext <= h[i] * (1 + 1e-12))
        assert np.all(ext >= h[i] * 0.999)
    # axis-aligned special case: the half extents are sigma * scale
    h0 = oc.support_half_extent(np.log([[0.1, 0.2, 0.3]]), [[2.0, 0, 0, 0]], 3.0)
    np.testing.assert_allclose(h0, [[0.3, 0.6, 0.9]], rtol=1e-14)
    # a quarter turn about z swaps the x and y extents
    h1 = oc.support_half_extent(np.log([[0.1, 0.2, 0.3]]), [[np.sqrt(0.5), 0, 0, np.sqrt(0.5)]], 3.0)
    np.testing.assert_allclose(h1, [[0.6, 0.3, 0.9]], rtol=1e-12)


def test_rotation_matches_the_projection_oracle():
    """The covariance used for the support is the one the projection oracle uses: for a camera with R = I the
    2-D covariance of a Gaussian on the optical axis is (f/z)^2 * Sigma[:2,:2] + dilation (EWA with x = y = 0)."""
    rng = np.random.default_rng(9)
    q = rng.standard_normal((1, 4)); ls = rng.normal(-2.0, 0.3, (1, 3))
    Sg = oc.covariance(ls, q)[0]
    cam = simple_camera(64, 150.0)
    p = gaussians([[0.0, 0.0, 5.0]], np.exp(ls), q, [0.0], [[0.5, 0.5, 0.5]])
    pr = oracle.project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], 0, cam.as_array())
    a, b, c = pr.conic_opacity[0, :3]
    cov2 = np.linalg.inv(np.array([[a, b], [b, c]]))
    want = (150.0 / 5.0) ** 2 * Sg[:2, :2] + 0.3 * np.eye(2)
    np.testing.assert_allclose(cov2, want, rtol=1e-9)


def test_cross_sets_closed_boxes_and_own_partition():
    lo = np.array([[-2.0, -2, 0], [0, -2, 0], [5, 5, 5]]); hi = np.array([[0.0, 2, 4], [2, 2, 4], [6, 6, 6]])
    mean = np.array([[-0.5, 0, 1], [-0.3, 0, 1], [-0.31, 0, 1], [-1.0, 0, 1]])
    ls = np.log(np.full((4, 3), 0.1)); q = np.tile([1.0, 0, 0, 0], (4, 1))
    member, margin = oc.cross_sets(mean, ls, q, 0, lo, hi, 3.0)
    # 3 sigma = 0.3: the Gaussian at x = -0.3 touches box 1 (closed), the one at -0.31 does not
    assert member[:, 1].tolist() == [False, True, False, False]
    assert not member[:, 0].any() and not member[:, 2].any()
    np.testing.assert_allclose(margin[1, 1], 0.0, atol=1e-12)
    np.testing.assert_allclose(margin[0, 1], -0.2, atol=1e-12)


def test_depth_ranges_bound_sampled_box_points():
    from paper_2606_18588_b200 import scenes
    rng = np.random.default_rng(2)
    cam = scenes.aerial_camera(96, 80, 60.0, 30.0, 40.0, 30.0, (1.0, 2.0, 0.0)).as_array()
    lo = np.array([[-20.0, -20, 0], [0, -20, 0]]); hi = np.array([[0.0, 0, 8], [20, 0, 8]])
    zr = oc.depth_ranges(lo, hi, [cam], [0, 0])
    R = cam[:9].reshape(3, 3); t = cam[9:12]
    for k in range(2):
        pts = rng.uniform(lo[k], hi[k], (20000, 3))
        z = pts @ R[2] + t[2]
        assert z.min() >= zr[k, 0] and z.max() <= zr[k, 1]
        corners = np.array([[(hi if i & 1 else lo)[k, 0], (hi if i & 2 else lo)[k, 1], (hi if i & 4 else lo)[k, 2]] for i in range(8)])
        zc = corners @ R[2] + t[2]
        assert zr[k, 0] == zc.min() and zr[k, 1] == zc.max()
    assert oc.depth_ranges(lo, hi, [cam], [0, -1])[1].tolist() == [np.inf, -np.inf]


def _fig25():
    """Two side-by-side partitions seen along +z (boundary x = 0), four Gaussians at depths 3 < 4 < 5 < 6:
    G1, G3 in partition 0 (x < 0), G2, G4 in partition 1; only G3 is wide enough to reach across."""
    cam = simple_camera(128, 200.0)
    p0 = gaussians([[-0.009, 0, 3], [-0.1, 0, 5]], [[0.0025] * 3, [0.4, 0.4, 0.01]], [[1, 0, 0, 0]] * 2, [0.4, 0.4],
                   [[1, 0, 0], [0, 0, 1]])
    p1 = gaussians([[0.012, 0, 4], [0.018, 0, 6]], [[0.003] * 3, [0.005] * 3], [[1, 0, 0, 0]] * 2, [0.4, 0.4],
                   [[0, 1, 0], [1, 1, 0]])
    cell_lo = np.array([[-2.0, -2, 2], [0, -2, 2]]); cell_hi = np.array([[0.0, 2, 10], [2, 2, 10]])
    vis_lo = cell_lo - [[0, 0, 0], [0.2, 0, 0]]; vis_hi = cell_hi + [[0.2, 0, 0], [0, 0, 0]]
    return cam, [p0, p1], cell_lo, cell_hi, vis_lo, vis_hi


def _render(parts, cam, lists=None):
    c = cam.as_array(); W, H = cam.width, cam.height
    cts, ds, bins = [], [], []
    for k, p in enumerate(parts):
        pr = oracle.project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], 0, c)
        bn = oracle.bin_sort(pr.means2d, pr.radius, pr.depth, W, H)
        vals, ranges = (bn.vals, bn.ranges) if lists is None else lists(k, pr, bn)
        pa = oracle.render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, vals, ranges, W, H)
        cts.append(pa.ct); ds.append(pa.d); bins.append((vals, ranges))
    image = oracle.compose(np.stack(cts), np.stack(ds), (0.1, 0.2, 0.3))[0]
    return image, bins


def test_fig25_worked_example():
    cam, parts, cell_lo, cell_hi, vis_lo, vis_hi = _fig25()
    c = cam.as_array(); W, H = cam.width, cam.height
    TX = W // 16
    state, _, _ = ov.visible_regions(vis_lo, vis_hi, c)
    omega = (state & 1) == 0
    zr = oc.depth_ranges(vis_lo, vis_hi, [c], [0, 0])
    Fs = []

    def lists(k, pr, bn):
        member, _ = oc.cross_sets(parts[k]["mean"], parts[k]["log_scale"], parts[k]["quat"], k, cell_lo, cell_hi)
        F = oc.filter_sets(member, pr.depth, k, zr, [0, 0])
        Fs.append(F)
        _, v, r = oc.filter_lists(bn.keys, bn.vals, F, state, TX * (H // 16))
        return v, r

    filtered, fbins = _render(parts, cam, lists)
    # the paper's statements about the figure (tests/golden/fig25_cross_boundary.txt)
    import os
    gold = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "fig25_cross_boundary.txt")):
        if line.strip() and not line.startswith("#"):
            w = line.split()
            gold.setdefault(w[0], []).append(w[1:])
    part_of = {g: int(k) for g, k in gold["partition_of"]}
    assert part_of == {"G1": 0, "G2": 1, "G3": 0, "G4": 1}          # how _fig25 lays the scene out
    local = {"G1": 0, "G3": 1, "G2": 0, "G4": 1}                    # index inside the partition (by depth)
    in_cross = {g for (g,) in gold["q_cross"]}
    for g in part_of:                                               # only G3 is in Q_cross, against partition 1
        assert bool(Fs[part_of[g]][local[g]].any()) == (g in in_cross), g
    assert gold["removed"] == [["r2", "G3"]] and gold["retained"] == [["r1", "G3"]]
    assert gold["filtered_sequence"] == [["r2", "G1", "G2", "G4"]]
    assert Fs[0].tolist() == [[False, False], [False, True]] and not Fs[1].any()
    r1, r2 = (64, 24), (64, 64)                      # (row, column): r1 sees partition 0 only, r2 both
    t1, t2 = (r1[0] // 16) * TX + r1[1] // 16, (r2[0] // 16) * TX + r2[1] // 16
    assert omega[0, t1] and not omega[1, t1] and omega[0, t2] and omega[1, t2]
    v0, rg0 = fbins[0]
    assert 1 in v0[rg0[t1, 0]:rg0[t1, 1]]            # "retained for ray r1"
    assert 1 not in v0[rg0[t2, 0]:rg0[t2, 1]]        # "removed for ray r2"
    assert 0 in v0[rg0[t2, 0]:rg0[t2, 1]]            # G1 stays
    # "yielding the consistent global ordering G1-G2-G4": the filtered two-partition image at r2 is the exactly
    # depth-sorted single-partition render of those three Gaussians
    cat = lambda ps: {k: np.concatenate([p[k] for p in ps]) for k in ps[0]}
    take = lambda p, idx: {k: v[idx] for k, v in p.items()}
    three = cat([take(parts[0], [0]), parts[1]])
    ref3, _ = _render([three], cam)
    np.testing.assert_allclose(filtered[r2], ref3[r2], rtol=0, atol=1e-12)
    # the premise: unfiltered, the partitions interleave (G1-G3-G2-G4) and the image differs from the exactly
    # sorted render of all four; at r1 nothing is filtered and nothing interleaves
    unfiltered, _ = _render(parts, cam)
    ref4, _ = _render([cat(parts)], cam)
    assert np.abs(unfiltered[r2] - ref4[r2]).max() > 1e-2
    np.testing.assert_allclose(filtered[r1], ref4[r1], rtol=0, atol=1e-12)
    assert np.abs(ref4[r1] - np.array([0.1, 0.2, 0.3])).max() > 1e-2     # G3 does show at r1


def test_host_depth_ranges_match_the_oracle():
    """splx_cross_depth_ranges is a HOST computation of the product: checked here without a GPU."""
    from paper_2606_18588_b200 import binding, scenes
    cams = [scenes.aerial_camera(96, 80, 60.0, 30.0, 40.0, 30.0, (1.0, 2.0, 0.0)),
            scenes.aerial_camera(96, 80, 60.0, 25.0, 55.0, 200.0, (-3.0, 1.0, 0.0))]
    lo = np.array([[-20.0, -20, 0], [0, -20, 0], [-20, 0, 0], [0, 0, 0]], np.float32)
    hi = np.array([[0.0, 0, 8], [20, 0, 8], [0, 20, 8], [20, 20, 8]], np.float32)
    vop = [0, 1, -1, 1]
    plan = binding.Plan(cams, vop, None, False)
    got = binding.cross_depth_ranges(lo, hi, plan)
    ref = oc.depth_ranges(lo, hi, [c.as_array() for c in cams], vop)
    assert got.dtype == np.float32 and got.shape == (4, 2)
    assert got[2].tolist() == [np.inf, -np.inf]
    np.testing.assert_allclose(got[[0, 1, 3]], ref[[0, 1, 3]], rtol=1e-6)
    assert abs(got[1, 0] - got[0, 0]) > 1e-3          # the two views really differ
    with np.testing.assert_raises(binding.SplxError):
        binding.cross_depth_ranges(lo[:0], hi[:0], plan)
