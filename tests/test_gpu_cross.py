"""-m gpu parity tests of cross-boundary per-ray filtering (Fig. 25; readings DESIGN.md s32)
through the C ABI, against oracle/cross_boundary.py.  Integers (masks, lists, ranges) bit-exact with the
Q_cross decision teacher-forced where fp32 and fp64 may differ; images 1e-5, gradients 1e-3."""
import numpy as np
import pytest
import torch

import oracle
from oracle import cross_boundary as oc
from oracle import visibility as ov
from paper_2606_18588_b200 import binding, scenes
from tests import gpu_common as G
from tests.test_oracle_cross import _fig25

pytestmark = pytest.mark.gpu


def _bits(mask, K):
    m = mask.astype(np.uint64)
    return np.stack([(m >> np.uint64(s)) & np.uint64(1) for s in range(K)], 1).astype(bool)


def _setup(sc, cam_index=0):
    """Trainer with visibility boxes (3-sigma inflated) and cross-boundary filtering against the cell boxes
    (boxes of the means)."""
    tr = G.make_trainer(sc)
    vis = scenes.partition_aabbs(sc.params, sc.part_offsets)
    cell = scenes.partition_aabbs(sc.params, sc.part_offsets, inflate_sigma=0.0)
    tr.set_aabbs(*vis)
    tr.set_cross(*cell)
    torch.cuda.synchronize()
    return tr, vis, cell


@pytest.fixture(scope="module")
def aerial():
    return scenes.small_aerial()


def test_cross_sets_match_oracle(aerial):
    sc = aerial
    tr, vis, cell = _setup(sc)
    got = _bits(tr._cross.cpu().numpy().view(np.uint64), sc.K)
    n_cross = 0
    for k in range(sc.K):
        a, b = int(sc.part_offsets[k]), int(sc.part_offsets[k + 1])
        member, margin = oc.cross_sets(sc.params["mean"][a:b], sc.params["log_scale"][a:b], sc.params["quat"][a:b], k,
                                       cell[0], cell[1], 3.0)
        diff = got[a:b] != member
        # fp32 against fp64: only a decision within rounding of the boundary may differ
        assert np.all(np.abs(margin[diff]) < 1e-4), (k, np.abs(margin[diff]).max())
        assert diff.mean() < 1e-3
        assert not got[a:b, k].any()
        n_cross += int(member.sum())
    assert n_cross > 100, "the scene must have cross-boundary Gaussians"


def test_depth_ranges_match_oracle(aerial):
    sc = aerial
    cam = sc.cameras[0]
    lo, hi = scenes.partition_aabbs(sc.params, sc.part_offsets)
    vop = [0, -1, 0, 0]
    plan = binding.Plan([cam], vop, None, False)
    got = binding.cross_depth_ranges(lo, hi, plan)
    ref = oc.depth_ranges(lo, hi, [cam.as_array()], vop)
    assert got[1].tolist() == [np.inf, -np.inf]
    keep = [0, 2, 3]
    np.testing.assert_allclose(got[keep], ref[keep], rtol=1e-6)


def _oracle_lists(sc, tr, cam, vop, state, zr, pr):
    """Per partition: the oracle's filtered lists built from the GPU's projection and Q_cross masks (teacher-forced
    decisions), positions made global the way the product lays the lists out (partition after partition)."""
    K = sc.K
    ntiles = state.shape[1]
    bits = _bits(tr._cross.cpu().numpy().view(np.uint64), K)
    out, pos = [], 0
    for k in range(K):
        a, b = int(sc.part_offsets[k]), int(sc.part_offsets[k + 1])
        if vop[k] < 0:
            out.append(None)
            continue
        bn = oracle.bin_sort(pr.means2d[a:b], pr.radius[a:b], pr.depth[a:b], cam.width, cam.height)
        F = oc.filter_sets(bits[a:b], pr.depth[a:b], k, zr, vop)
        keys, vals, ranges = oc.filter_lists(bn.keys, bn.vals, F, state, ntiles)
        out.append((keys, vals, ranges, pos, bn.M))
        pos += len(vals)
    return out, pos


def test_filtered_binning_bit_exact(aerial):
    sc = aerial
    cam = sc.cameras[0]
    tr, vis, cell = _setup(sc)
    state, part = binding.visible_regions(vis[0], vis[1], cam)
    vop = [0 if (part >> k) & 1 else -1 for k in range(sc.K)]
    dev_state = torch.from_numpy(state.reshape(-1)).cuda()
    plan = tr.make_plan([cam], vop, dev_state, False)
    c = tr.ctx
    tr._workspaces(cam)
    c.project_plan(tr.params, tr.part_offsets, plan, tr.sh_degree, tr.proj)
    # unfiltered, for the count
    c.bin_sort_plan(tr.proj, tr.part_offsets, plan, tr.bins, tr._ws_sort)
    M0 = tr.num_intersections()
    tr._bin_sort(tr.proj, plan, tr.bins, tr._ws_sort)
    M1, keys1, vals1, ranges1 = G.gpu_bins(tr)
    pr = G.gpu_projected(tr)
    zr = binding.cross_depth_ranges(vis[0], vis[1], plan)
    lists, kept = _oracle_lists(sc, tr, cam, vop, state, zr, pr)
    assert M1 == kept and 0 < M0 - M1 < M0, (M0, M1, kept)
    ntiles = state.shape[1]
    for k in range(sc.K):
        if lists[k] is None:
            assert not ranges1[k].any()
            continue
        keys, vals, ranges, pos, _ = lists[k]
        a = int(sc.part_offsets[k])
        want = ov.apply_tile_state(ranges, state[k]).astype(np.int64)
        live = want[:, 1] > want[:, 0]
        assert np.array_equal(ranges1[k][live].astype(np.int64), want[live] + pos)
        assert not ranges1[k][~live].any()
        assert np.array_equal(vals1[pos:pos + len(vals)].astype(np.int64), vals.astype(np.int64) + a)
        assert np.array_equal(keys1[pos:pos + len(vals)] & np.uint64(0xffffffff), keys & np.uint64(0xffffffff))
        assert np.array_equal((keys1[pos:pos + len(vals)] >> np.uint64(32)).astype(np.int64),
                              (keys >> np.uint64(32)).astype(np.int64) + k * ntiles)


def test_zero_masks_change_nothing(aerial):
    sc = aerial
    cam = sc.cameras[0]
    tr, vis, cell = _setup(sc)
    plan = tr.make_plan([cam], None, None, False)
    c = tr.ctx
    tr._workspaces(cam)
    c.project_plan(tr.params, tr.part_offsets, plan, tr.sh_degree, tr.proj)
    c.bin_sort_plan(tr.proj, tr.part_offsets, plan, tr.bins, tr._ws_sort)
    M0, k0, v0, r0 = G.gpu_bins(tr)
    k0, v0, r0 = k0.copy(), v0.copy(), r0.copy()
    tr._cross.zero_()
    tr._bin_sort(tr.proj, plan, tr.bins, tr._ws_sort)
    M1, k1, v1, r1 = G.gpu_bins(tr)
    assert M1 == M0 and np.array_equal(k1, k0) and np.array_equal(v1, v0) and np.array_equal(r1, r0)


def test_filtered_iteration_matches_oracle(aerial):
    """Forward image and parameter gradients of a whole iteration with the filter on: the later stages see only the
    filtered lists, exactly as the oracle's stages do when handed the oracle's filtered lists."""
    sc = aerial
    cam = sc.cameras[0]
    c64 = cam.as_array()
    W, H = cam.width, cam.height
    tr, vis, cell = _setup(sc)
    state, part = binding.visible_regions(vis[0], vis[1], cam)
    vop = [0] * sc.K
    assert part == (1 << sc.K) - 1
    dev_state = torch.from_numpy(state.reshape(-1)).cuda()
    plan = tr.make_plan([cam], vop, dev_state, True)
    target = torch.from_numpy(sc.targets[0]).cuda()[None]
    img = G.np32(tr.forward_plan(plan))[0].astype(np.float64)
    tr.loss_grad_plan(target)
    tr.backward_plan(overwrite=True)
    torch.cuda.synchronize()
    zr = binding.cross_depth_ranges(vis[0], vis[1], plan)
    bits = _bits(tr._cross.cpu().numpy().view(np.uint64), sc.K)
    ntiles = state.shape[1]
    parts, prs, bins, pas = [], [], [], []
    for k in range(sc.K):
        a, b = int(sc.part_offsets[k]), int(sc.part_offsets[k + 1])
        p = {key: sc.params[key][a:b].astype(np.float64) for key in scenes.PARAM_KEYS}
        pr = oracle.project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], sc.sh_degree, c64)
        bn = oracle.bin_sort(pr.means2d, pr.radius, pr.depth, W, H)
        F = oc.filter_sets(bits[a:b], pr.depth, k, zr, vop)
        _, vals, ranges = oc.filter_lists(bn.keys, bn.vals, F, state, ntiles)
        ranges = ov.apply_tile_state(ranges, state[k])
        pa = oracle.render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, vals, ranges, W, H)
        parts.append(p); prs.append(pr); bins.append((vals, ranges)); pas.append(pa)
    ct = np.stack([pa.ct for pa in pas]); d = np.stack([pa.d for pa in pas])
    image, T_total, order, order_margin = oracle.compose(ct, d, sc.bg)
    frag = np.zeros((H, W), bool)
    for pa in pas:
        frag |= pa.margin < G.FRAGILE_MARGIN
    frag |= order_margin < 1e-6
    ok = G.close(img, image).all(axis=2)
    assert ok[~frag].all() and frag.mean() < 0.02, (int((~ok & ~frag).sum()), frag.mean())
    assert np.abs(img - image).max() < G.FRAGILE_TOL
    # the filter did something to the picture
    tr.set_cross(None, None)
    img_off = G.np32(tr.forward_plan(plan))[0].astype(np.float64)
    assert np.abs(img_off - img).max() > 1e-3
    _, g_image = oracle.l1(image, sc.targets[0].astype(np.float64))
    g_ct = oracle.compose_bwd(ct, d, g_image, sc.bg)
    ref = []
    for k in range(sc.K):
        p, pr = parts[k], prs[k]
        vals, ranges = bins[k]
        g2 = oracle.raster_bwd(pr.means2d, pr.conic_opacity, pr.rgb, vals, ranges, W, H, g_ct[k])
        ref.append(oracle.project_bwd(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], sc.sh_degree, c64,
                                      pr.radius, pr.clamp, *g2))
    for key in scenes.PARAM_KEYS:
        got = G.np32(tr.grads[key]).astype(np.float64).reshape(-1)
        want = np.concatenate([g[key].reshape(-1) for g in ref])
        assert G.rel_l2(got, want) <= 1e-3, (key, G.rel_l2(got, want))
        assert G.grad_close(got, want) <= G.GRAD_MAX_TOL, (key, G.grad_close(got, want))


def test_fig25_on_the_gpu():
    """The worked example of Fig. 25 through the C ABI: G3 leaves the list of r2's tile, stays in r1's, and the image
    at r2 is the oracle's filtered one."""
    cam, parts, cell_lo, cell_hi, vis_lo, vis_hi = _fig25()
    params = {k: np.concatenate([p[k] for p in parts]).astype(np.float32) for k in scenes.PARAM_KEYS}
    offs = np.array([0, 2, 4], np.int64)
    from paper_2606_18588_b200.engine import Trainer
    tr = Trainer(params, offs, cam.width, cam.height, 0, (0.1, 0.2, 0.3))
    tr.set_aabbs(vis_lo, vis_hi)
    tr.set_cross(cell_lo, cell_hi)
    mask = tr._cross.cpu().numpy().view(np.uint64)
    assert mask.tolist() == [0, 2, 0, 0]
    state, part = binding.visible_regions(vis_lo, vis_hi, cam)
    plan = tr.make_plan([cam], [0, 0], torch.from_numpy(state.reshape(-1)).cuda(), True)
    img = G.np32(tr.forward_plan(plan))[0].astype(np.float64)
    M, keys, vals, ranges = G.gpu_bins(tr)
    TX = cam.width // 16
    t1, t2 = (64 // 16) * TX + 24 // 16, (64 // 16) * TX + 64 // 16
    assert 1 in vals[ranges[0, t1, 0]:ranges[0, t1, 1]]
    assert 1 not in vals[ranges[0, t2, 0]:ranges[0, t2, 1]] and 0 in vals[ranges[0, t2, 0]:ranges[0, t2, 1]]
    # oracle: same chain in fp64
    c = cam.as_array()
    zr = oc.depth_ranges(vis_lo, vis_hi, [c], [0, 0])
    cts, ds = [], []
    for k, p in enumerate(parts):
        pr = oracle.project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], 0, c)
        bn = oracle.bin_sort(pr.means2d, pr.radius, pr.depth, cam.width, cam.height)
        member, _ = oc.cross_sets(p["mean"], p["log_scale"], p["quat"], k, cell_lo, cell_hi)
        F = oc.filter_sets(member, pr.depth, k, zr, [0, 0])
        _, v, r = oc.filter_lists(bn.keys, bn.vals, F, state, state.shape[1])
        pa = oracle.render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, v, ov.apply_tile_state(r, state[k]),
                                   cam.width, cam.height)
        cts.append(pa.ct); ds.append(pa.d)
    ref = oracle.compose(np.stack(cts), np.stack(ds), (0.1, 0.2, 0.3))[0]
    assert G.close(img[64, 64], ref[64, 64]).all() and G.close(img[64, 24], ref[64, 24]).all()
    assert np.mean(G.close(img, ref).all(axis=2)) > 0.999
