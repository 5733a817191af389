"""-m gpu parity tests of the two optional subsystems through the C ABI (the *_plan calls): visibility
prediction and conflict-free consolidation of B views (L247-L249), against
oracle/visibility.py.  Same bars as the core: integers bit-exact, images 1e-5, gradients 1e-3."""
import numpy as np
import pytest
import torch

import oracle
from oracle import visibility as ov
from paper_2606_18588_b200 import binding, scenes
from tests import gpu_common as G

pytestmark = pytest.mark.gpu


def _trainer(sc):
    tr = G.make_trainer(sc)
    tr.set_aabbs(*scenes.partition_aabbs(sc.params, sc.part_offsets))
    return tr


def _grads_np(tr):
    return {k: G.np32(tr.grads[k]).astype(np.float64) for k in scenes.PARAM_KEYS}


def _check_grads(tr, ref_grads, res=None):
    G.check_grads(tr, ref_grads, res)


def _fragile(res):
    frag = np.zeros(res.image.shape[:2], bool)
    for pa in res.partials:
        frag |= pa.margin < G.FRAGILE_MARGIN
    if res.order_margin is not None:
        frag |= res.order_margin < 1e-6
    return frag


@pytest.fixture(scope="module")
def aerial():
    return scenes.small_aerial()


@pytest.fixture(scope="module")
def city():
    return scenes.small_city()       # every view sees every partition; opaque: saturation everywhere


@pytest.fixture(scope="module")
def blocks():
    return scenes.small_blocks()     # a view sees 2-4 of the 8 partitions: conflict-free buckets exist


def test_sparse_partials_change_nothing(aerial):
    """SPLX_PLAN_SPARSE only avoids storing and loading identity partials: image bit-equal, gradients equal."""
    sc = aerial
    cam = sc.cameras[0]
    target = torch.from_numpy(sc.targets[0]).cuda()[None]
    out = []
    for sparse in (False, True):
        tr = _trainer(sc)
        tr.partials.ct.fill_(float("nan")); tr.partials.d.fill_(float("nan"))   # unread slots may hold anything
        plan = tr.make_plan([cam], None, None, sparse)
        img = tr.forward_plan(plan).clone()
        tr.loss_grad_plan(target)
        tr.backward_plan(overwrite=True)
        torch.cuda.synchronize()
        out.append((img, _grads_np(tr), tr))
    assert torch.equal(out[0][0], out[1][0])
    assert not torch.isnan(out[1][0]).any()
    for key in scenes.PARAM_KEYS:
        assert G.grad_close(out[1][1][key], out[0][1][key]) <= 1e-4, key
    # and the dense plan is the single-view call
    tr = out[0][2]
    tr.forward(cam)
    assert torch.equal(tr.image, out[0][0][0])


def test_geometric_state_and_masked_binning(city):
    """splx_visible_regions == LP oracle on the scene's own boxes; bin_sort under the state keeps keys/vals and
    zeroes exactly the ranges of the skipped slots (bit-exact, teacher-forced)."""
    sc = city
    cam = sc.cameras[1]
    lo, hi = scenes.partition_aabbs(sc.params, sc.part_offsets, inflate_sigma=0.0)   # tight boxes: some lists are cut
    tr = G.make_trainer(sc)
    state, part = binding.visible_regions(lo, hi, cam)
    ref, part_ref, margin = ov.visible_regions(lo, hi, cam.as_array())
    robust = np.abs(margin) > 1e-6
    assert np.array_equal(state[robust], ref[robust]) and part == part_ref and robust.mean() > 0.98
    assert 0 < (state == 0).mean() < 1
    vop = [0 if (part >> k) & 1 else -1 for k in range(sc.K)]
    dev_state = torch.from_numpy(state.reshape(-1)).cuda()
    c = tr.ctx
    tr._workspaces(cam)
    # unmasked reference binning on the GPU
    plan0 = tr.make_plan([cam], vop, None, False)
    c.project_plan(tr.params, tr.part_offsets, plan0, tr.sh_degree, tr.proj)
    c.bin_sort_plan(tr.proj, tr.part_offsets, plan0, tr.bins, tr._ws_sort)
    M0, keys0, vals0, ranges0 = G.gpu_bins(tr)
    keys0, vals0, ranges0 = keys0.copy(), vals0.copy(), ranges0.copy()
    plan1 = tr.make_plan([cam], vop, dev_state, False)
    c.bin_sort_plan(tr.proj, tr.part_offsets, plan1, tr.bins, tr._ws_sort)
    M1, keys1, vals1, ranges1 = G.gpu_bins(tr)
    assert M1 == M0 and np.array_equal(keys1, keys0) and np.array_equal(vals1, vals0)
    n_cut = 0
    pr = G.gpu_projected(tr)
    pos = 0
    for k in range(sc.K):
        a, b = tr.part_offsets[k], tr.part_offsets[k + 1]
        if vop[k] < 0:
            assert not ranges1[k].any()
            continue
        bn = oracle.bin_sort(pr.means2d[a:b], pr.radius[a:b], pr.depth[a:b], cam.width, cam.height)
        want = ov.apply_tile_state(bn.ranges, state[k]).astype(np.int64)
        live = want[:, 1] > want[:, 0]
        assert np.array_equal(ranges1[k][live].astype(np.int64), want[live] + pos)
        assert not ranges1[k][~live].any()
        n_cut += int(((bn.ranges[:, 1] > bn.ranges[:, 0]) & ~live).sum())
        pos += bn.M
    assert pos == M1 and n_cut > 0, "tight boxes must cut some boundary lists"


def test_non_participants_are_skipped_and_cleared(blocks):
    """A partition with view -1 is not projected (its projected rows keep stale values), gets no keys, and
    SPLX_PB_OVERWRITE writes zeros into its gradient rows."""
    sc = blocks
    cam = sc.cameras[1]
    tr = _trainer(sc)
    part = tr.participants(1, cam)
    vop = [0 if (part >> k) & 1 else -1 for k in range(sc.K)]
    assert 0 < sum(v == 0 for v in vop) < sc.K
    tr.proj.tiles_touched.fill_(7); tr.proj.radius.fill_(9)
    for v in tr.grads.values():
        v.fill_(5.0)
    plan = tr.make_plan([cam], vop, None, True)
    tr.forward_plan(plan)
    tr.loss_grad_plan(torch.from_numpy(sc.targets[0]).cuda()[None])
    tr.backward_plan(overwrite=True)
    torch.cuda.synchronize()
    tt = G.u32(tr.proj.tiles_touched)
    vals = G.u32(tr.bins.vals)[:tr.num_intersections()]
    for k in range(sc.K):
        a, b = tr.part_offsets[k], tr.part_offsets[k + 1]
        inside = ((vals >= a) & (vals < b)).sum()
        if vop[k] < 0:
            assert (tt[a:b] == 7).all() and inside == 0
            for key in scenes.PARAM_KEYS:
                w = scenes.PARAM_WIDTH[key]
                assert not G.np32(tr.grads[key])[a * w:b * w].any(), key
        else:
            assert (tt[a:b] != 7).any()
    # against the oracle on the participating partitions only, and against the oracle on ALL partitions: the
    # boxes contain every 3-sigma support, so dropping the non-participants changes nothing
    views, grads = ov.iteration_plan(sc.partitions(), [cam.as_array()], vop, sc.sh_degree, [sc.targets[0]], sc.bg)
    res_all = oracle.forward(sc.partitions(), cam.as_array(), sc.sh_degree, sc.bg)
    assert np.array_equal(res_all.image, views[0].image)
    frag = _fragile(views[0])
    img = G.np32(tr._images[0]).astype(np.float64)
    assert (G.close(img, views[0].image).all(-1) | frag).mean() >= 1 - 1e-4
    _check_grads(tr, grads)


def test_saturation_detection_teacher_forced(city):
    """compose's tile_state_out against the oracle's front products computed from the GPU's own partials."""
    sc = city
    cam = sc.cameras[0]
    for eps in (1e-4, 1e-2):
        tr = _trainer(sc)
        part = tr.participants(0, cam)
        vop = [0 if (part >> k) & 1 else -1 for k in range(sc.K)]
        members = [k for k in range(sc.K) if vop[k] == 0]
        geom = tr._geom_state[0]
        state_dev = torch.from_numpy(geom.reshape(-1).copy()).cuda()
        plan = tr.make_plan([cam], vop, state_dev, False)          # dense: every participant's partial is stored
        out = torch.full_like(state_dev, 77)
        tr.forward_plan(plan, eps, out)
        torch.cuda.synchronize()
        ct = G.np32(tr.partials.ct).astype(np.float64); d = G.np32(tr.partials.d).astype(np.float64)
        ref, margin = ov.saturation(ct, d, eps, geom, members)
        got = G.np32(out).reshape(sc.K, -1)
        for k in range(sc.K):
            if vop[k] < 0:
                assert (got[k] == 77).all()          # rows of non-participants are not touched
                continue
            robust = margin[k] > 1e-5
            assert np.array_equal(got[k][robust], ref[k][robust]), (eps, k)
            assert robust.mean() > 0.99
        if eps == 1e-2:
            assert (ref[members] & ov.TILE_SATURATED).any(), "the city scene must saturate somewhere at eps = 1e-2"


def test_consolidated_bucket_against_the_oracle(blocks):
    """B views of a conflict-free bucket in ONE launch per stage: images per view and the summed gradients
    against the oracle's plan iteration, and against the same views run one by one on the GPU."""
    sc = blocks
    tr = _trainer(sc)
    ids = list(range(len(sc.cameras)))
    groups = tr.buckets(ids, sc.cameras, consolidate=True)
    parts = [tr.participants(v, sc.cameras[v]) for v in ids]
    ref_b, nb = ov.schedule_views(parts)
    assert [sorted(g) for g in groups] == [sorted(i for i in ids if ref_b[i] == b) for b in range(nb)]
    multi = [g for g in groups if len(g) > 1]
    assert multi, "the test scene must have a bucket with more than one view"
    grp = multi[0]
    cams = [sc.cameras[i] for i in grp]
    plan, _ = tr.bucket_plan(grp, cams, saturation=False)
    targets = torch.from_numpy(np.stack([sc.targets[i] for i in grp])).cuda()
    imgs = tr.forward_plan(plan).clone()
    tr.loss_grad_plan(targets)
    tr.backward_plan(overwrite=True)
    torch.cuda.synchronize()
    state = G.np32(plan.tile_state).reshape(sc.K, -1)
    views, grads = ov.iteration_plan(sc.partitions(), [c.as_array() for c in cams], plan.view_of_part, sc.sh_degree,
                                     [sc.targets[i] for i in grp], sc.bg, tile_state=state)
    for j, res in enumerate(views):
        frag = _fragile(res)
        img = G.np32(imgs[j]).astype(np.float64)
        ok = G.close(img, res.image).all(-1)
        assert (~(ok | frag)).sum() <= 1e-4 * frag.size, j
        assert np.abs(img - res.image).max() <= G.FRAGILE_TOL
    _check_grads(tr, grads)
    g_multi = _grads_np(tr)
    # the same views one after the other (one-view plans, gradients accumulated): same images, same sum
    tr2 = _trainer(sc)
    for j, i in enumerate(grp):
        vop = [0 if plan.view_of_part[k] == j else -1 for k in range(sc.K)]
        p1 = tr2.make_plan([sc.cameras[i]], vop, plan.tile_state, True)
        img1 = tr2.forward_plan(p1)
        assert torch.equal(img1[0], imgs[j])
        tr2.loss_grad_plan(targets[j:j + 1])
        tr2.backward_plan(overwrite=(j == 0))
    torch.cuda.synchronize()
    g_seq = _grads_np(tr2)
    for key in scenes.PARAM_KEYS:
        assert G.grad_close(g_multi[key], g_seq[key]) <= 1e-4, key


@pytest.mark.parametrize("case", ["aerial_eps_1e-2", "street_eps_1e-4"])
def test_iteration_views_with_visibility_prediction(city, case):
    """The whole subsystem: two iterations over B views; the second applies the saturated tiles the first
    detected.  Every skipped slot has (oracle) front product < eps, and the image stays within eps * max rgb of
    the oracle that skips nothing (SURVEY s8(f) agreement rule).  Second case: the paper's own threshold eps = 1e-4
    (L353) on street-level views of the same recipe (walls of two partitions stand in front of a third: L296), where the
    literal test of L213 does fire."""
    if case == "aerial_eps_1e-2":
        sc, eps = city, 1e-2
    else:
        sc = scenes.city(n=30_000, width=320, height=176, extent=120.0, n_buildings=12, grid=(4, 2), altitude=35.0,
                         height_range=(5.0, 25.0), n_views=4, street=True, name="street_30000")
        eps = 1e-4
    tr = _trainer(sc)
    ids = list(range(len(sc.cameras)))
    targets = torch.from_numpy(np.stack(sc.targets)).cuda()
    lr0 = dict(tr.lr)
    tr.lr = {k: 0.0 for k in lr0}          # keep the parameters fixed so that both iterations see the same scene
    n_launch = tr.iteration_views(ids, sc.cameras, targets, sat_eps=eps)
    assert n_launch == len(tr.buckets(ids, sc.cameras))
    # second visit: saturated slots are skipped
    groups = tr.buckets(ids, sc.cameras)
    skipped = 0
    for grp in groups:
        cams = [sc.cameras[i] for i in grp]
        plan, state_out = tr.bucket_plan(grp, cams)
        state = G.np32(plan.tile_state).reshape(sc.K, -1).copy()
        imgs = tr.forward_plan(plan, eps, state_out).clone()
        torch.cuda.synchronize()
        full, _ = ov.iteration_plan(sc.partitions(), [c.as_array() for c in cams], plan.view_of_part, sc.sh_degree,
                                    [sc.targets[i] for i in grp], sc.bg)
        for j, res in enumerate(full):
            members = res.members
            ct = np.stack([p.ct for p in res.partials]); d = np.stack([p.d for p in res.partials])
            front = ov.front_products(ct, res.order)
            TX = (cams[j].width + 15) // 16
            for jj, k in enumerate(members):
                for t in np.nonzero(state[k] & ov.TILE_SATURATED)[0]:
                    x0, y0 = (t % TX) * 16, (t // TX) * 16
                    assert np.all(front[jj, y0:y0 + 16, x0:x0 + 16] < eps * (1 + 1e-3)), (k, t)
                    skipped += 1
            rgb_max = max(float(p.rgb.max()) for p in res.proj)
            frag = _fragile(res)
            img = G.np32(imgs[j]).astype(np.float64)
            err = np.abs(img - res.image).max(-1)
            assert (err[~frag] <= eps * rgb_max + 1e-5).all()
    assert skipped > 0


def test_step_host_equals_the_stage_calls(aerial):
    """Trainer.step_host (the end-to-end call bench.py times: host buffers, copies overlapped on a side stream)
    produces the image, loss and parameter update of the plain stage-by-stage iteration."""
    sc = aerial
    cam = sc.cameras[0]
    a, b = _trainer(sc), _trainer(sc)
    tgt_host = torch.from_numpy(sc.targets[0]).pin_memory()
    img_host = torch.empty((cam.height, cam.width, 3), dtype=torch.float32).pin_memory()
    loss_host = torch.zeros(2, dtype=torch.float64).pin_memory()
    target = torch.from_numpy(sc.targets[0]).cuda()
    for it in range(2):
        a.step_host(0, cam, tgt_host, img_host, loss_host)
        b.loss_sum.zero_()
        b.forward(cam)
        b.loss_grad(target)
        b.backward(overwrite=True)
        b.adam_step()
        torch.cuda.synchronize()
        if it == 0:   # same parameters in: bit-equal image (later steps differ by the atomics' summation order)
            assert torch.equal(img_host.cuda(), b.image)
            assert float(loss_host[0].item()) == pytest.approx(float(b.loss_sum[0].item()), rel=1e-6)   # fused loss: other summation order
        else:
            assert torch.allclose(img_host.cuda(), b.image, rtol=0, atol=1e-5)
            assert float(loss_host[0].item()) == pytest.approx(float(b.loss_sum[0].item()), rel=1e-6)
    for key in scenes.PARAM_KEYS:
        assert torch.allclose(a.params[key], b.params[key], rtol=1e-3, atol=1e-6), key


def test_fused_compose_loss_backward_equals_the_staged_calls(blocks):
    """splx_compose_l1_backward_plan (a6 + a7 + a8 in one kernel) against the three staged calls on a two-view
    bucket: image, T_total, dL/dC^k, dL/dT^k and the saturation bytes bit-equal, the loss to rounding."""
    sc = blocks
    tr = _trainer(sc)
    grp = [0, 3]
    cams = [sc.cameras[i] for i in grp]
    plan, state = tr.bucket_plan(grp, cams)
    targets = torch.from_numpy(np.stack([sc.targets[i] for i in grp])).cuda()
    c = tr.ctx
    st_a = state.clone(); st_b = state.clone()
    imgs = tr.forward_plan(plan, 1e-2, st_a).clone()
    T_a = tr._T_totals[:2].clone()
    tr.loss_sum.zero_()
    tr.loss_grad_plan(targets)
    loss_a = float(tr.loss_sum[0].item())
    g_ct_a = torch.zeros((sc.K, cams[0].height, cams[0].width, 4), device="cuda")
    c.compose_backward_plan(tr.partials, tr.bins, plan, tr.bg, tr._g_images[:2], None, g_ct_a)
    g_ct_b = torch.zeros_like(g_ct_a)
    img_b = torch.empty_like(imgs); T_b = torch.empty_like(T_a)
    tr.loss_sum.zero_()
    c.compose_l1_backward_plan(tr.partials, tr.bins, plan, tr.bg, targets, img_b, T_b, tr.loss_sum, g_ct_b, scale=2.0,
                               sat_eps=1e-2, tile_state_out=st_b)
    torch.cuda.synchronize()
    assert torch.equal(img_b, imgs) and torch.equal(T_b, T_a)
    assert torch.equal(g_ct_b, g_ct_a)
    assert torch.equal(st_a, st_b)
    assert float(tr.loss_sum[0].item()) == pytest.approx(loss_a, rel=1e-6)
    assert g_ct_a.abs().max() > 0


def test_kd_partitions_under_the_plan():
    """The paper's own partitioner (KD median splits, L480) instead of the uniform grid: the plan path takes any
    boxes.  One view, geometric state from the KD cells' 3-sigma boxes, against the oracle."""
    sc = scenes.aerial(n=20_000, width=320, height=176, grid=(2, 2), log_scale_mu=-0.9, partition="kd", name="aerial_kd")
    assert scenes.imbalance_ratio(sc.part_offsets) < 1e-3
    cam = sc.cameras[0]
    tr = _trainer(sc)
    plan, _ = tr.bucket_plan([0], [cam], saturation=False)
    target = torch.from_numpy(sc.targets[0]).cuda()[None]
    imgs = tr.iteration_fused(plan, target, overwrite=True).clone()
    torch.cuda.synchronize()
    state = G.np32(plan.tile_state).reshape(sc.K, -1)
    views, grads = ov.iteration_plan(sc.partitions(), [cam.as_array()], plan.view_of_part, sc.sh_degree, [sc.targets[0]],
                                     sc.bg, tile_state=state)
    frag = _fragile(views[0])
    ok = G.close(G.np32(imgs[0]).astype(np.float64), views[0].image).all(-1)
    assert (~(ok | frag)).sum() <= 1e-4 * frag.size
    _check_grads(tr, grads, views[0])
    full = oracle.forward(sc.partitions(), cam.as_array(), sc.sh_degree, sc.bg)     # no state at all
    assert np.array_equal(full.image, views[0].image)


def test_projection_backward_over_the_visible_list(blocks):
    """splx_project_backward_list_plan (+= over the binning's list of visible Gaussians) == the dense += call:
    a culled Gaussian has no gradient, so only the rows touched differ, not the result."""
    sc = blocks
    cam = sc.cameras[1]
    rng = np.random.default_rng(51)
    a, b = _trainer(sc), _trainer(sc)
    part = a.participants(1, cam)
    vop = [0 if (part >> k) & 1 else -1 for k in range(sc.K)]
    g2d = np.zeros((a.n, 12), np.float32)
    g2d[:, :9] = rng.standard_normal((a.n, 9))
    old = rng.standard_normal(a.flat["grad"].shape).astype(np.float32)
    for tr in (a, b):
        plan = tr.make_plan([cam], vop, None, True)
        tr._workspaces(cam)
        tr.ctx.project_plan(tr.params, tr.part_offsets, plan, tr.sh_degree, tr.proj)
        tr.ctx.bin_sort_plan(tr.proj, tr.part_offsets, plan, tr.bins, tr._ws_sort)
        tr.flat["grad"].copy_(torch.from_numpy(old))
        tr._plan = plan
    ga, gb = torch.from_numpy(g2d).cuda(), torch.from_numpy(g2d).cuda()
    a.ctx.project_backward_plan(a.params, a.part_offsets, a._plan, a.sh_degree, a.proj, ga, a.grads, clear_g2d=True)
    lst, cnt = b.ctx.bin_sort_visible(b._ws_sort, b.n, b.capacity, b.K, cam)
    b.ctx.project_backward_list_plan(b.params, b.part_offsets, b._plan, b.sh_degree, b.proj, gb, b.grads, lst, cnt,
                                     clear_g2d=True)
    torch.cuda.synchronize()
    assert torch.equal(a.flat["grad"], b.flat["grad"])
    assert torch.equal(ga, gb)
    assert not torch.equal(a.flat["grad"], torch.from_numpy(old).cuda())
    n_vis = int((b.proj.radius[torch.as_tensor([i for k in range(sc.K) if vop[k] == 0
                                                  for i in range(b.part_offsets[k], b.part_offsets[k + 1])]).cuda()] > 0).sum())
    assert 0 < n_vis < b.n


def test_projection_in_two_halves_equals_the_single_call(blocks):
    """splx_project_geometry_plan + (after the binning) splx_project_colour_list_plan == splx_project_plan: identical
    bytes in every output of the participating partitions, the colour compared on the visible Gaussians (a culled
    one has none), and the binning built on the geometry alone is the same binning."""
    sc = blocks
    cam = sc.cameras[1]
    a, b = _trainer(sc), _trainer(sc)
    part = a.participants(1, cam)
    vop = [0 if (part >> k) & 1 else -1 for k in range(sc.K)]
    for tr in (a, b):
        tr._plan = tr.make_plan([cam], vop, None, True)
        tr._workspaces(cam)
        for t in (tr.proj.rgb, tr.proj.blend):
            t.fill_(-7.0)
        tr.proj.clamp.fill_(9)
    a.ctx.project_plan(a.params, a.part_offsets, a._plan, a.sh_degree, a.proj)
    a.ctx.bin_sort_plan(a.proj, a.part_offsets, a._plan, a.bins, a._ws_sort)
    b.ctx.project_geometry_plan(b.params, b.part_offsets, b._plan, b.proj)
    b.ctx.bin_sort_plan(b.proj, b.part_offsets, b._plan, b.bins, b._ws_sort)
    lst, cnt = b.ctx.bin_sort_visible(b._ws_sort, b.n, b.capacity, b.K, cam)
    b.ctx.project_colour_list_plan(b.params, b.part_offsets, b._plan, b.sh_degree, b.proj, lst, cnt)
    torch.cuda.synchronize()
    rows = torch.as_tensor([i for k in range(sc.K) if vop[k] == 0 for i in range(a.part_offsets[k], a.part_offsets[k + 1])]).cuda()
    vis = rows[a.proj.radius[rows] > 0]
    assert 0 < vis.numel() < a.n
    for name in ("radius", "tiles_touched"):
        assert torch.equal(getattr(a.proj, name)[rows], getattr(b.proj, name)[rows]), name
    for name in ("means2d", "depth", "conic_opacity", "rgb", "clamp", "blend"):
        x, y = getattr(a.proj, name), getattr(b.proj, name)
        x, y = x.view(a.n, -1)[vis], y.view(b.n, -1)[vis]
        assert torch.equal(x.view(torch.uint8), y.view(torch.uint8)), name
    m = int(a.bins.num_intersections[0])
    assert m == int(b.bins.num_intersections[0]) and m > 0
    assert torch.equal(a.bins.keys[:m], b.bins.keys[:m]) and torch.equal(a.bins.vals[:m], b.bins.vals[:m])


def test_pipelined_buckets_equal_the_sequential_iteration(city):
    """Multi-bucket iterations project and sort bucket g+1 on a second stream while bucket g is blended (double-buffered
    projected / binning sets): same gradients, same saturation bytes, same parameters as one bucket after the other."""
    sc = city
    ids = list(range(len(sc.cameras)))
    targets = torch.from_numpy(np.stack(sc.targets)).cuda()
    out = []
    for pipe in (False, True):
        tr = _trainer(sc)
        tr.pipeline_buckets = pipe
        for _ in range(3):
            n_b = tr.iteration_views(ids, sc.cameras, targets, sat_eps=1e-2)
        torch.cuda.synchronize()
        assert n_b > 1
        states = {k: v.clone() for k, v in tr._bucket_state.items()}
        out.append((tr.flat["grad"].clone(), tr.flat["param"].clone(), states))
    g0, g1 = out[0][0], out[1][0]
    assert float((g0 - g1).abs().max()) <= 1e-4 * float(g0.abs().max())
    close = (out[0][1] - out[1][1]).abs() <= 1e-3 * out[0][1].abs() + 2e-6
    assert close.float().mean().item() > 0.999
    for k in out[0][2]:
        assert (out[0][2][k] != out[1][2][k]).float().mean().item() < 1e-3, k     # a slot within rounding of eps may flip


def test_iteration_views_gradients_against_the_oracle(blocks):
    """A whole multi-bucket iteration (two consolidated two-view buckets + two single views; first bucket '=', later
    buckets '+=' over the visible list with per-row cameras; pipelined over two streams): the accumulated gradient
    against the sum of the oracle's plan iterations."""
    sc = blocks
    tr = _trainer(sc)
    tr.lr = {k: 0.0 for k in tr.lr}
    ids = list(range(len(sc.cameras)))
    targets = torch.from_numpy(np.stack(sc.targets)).cuda()
    groups = tr.buckets(ids, sc.cameras)
    assert any(len(g) > 1 for g in groups[1:]), "a consolidated bucket must take the accumulating path"
    tr.iteration_views(ids, sc.cameras, targets, saturation=False)
    torch.cuda.synchronize()
    total = None
    for grp in groups:
        cams = [sc.cameras[i] for i in grp]
        plan, _ = tr.bucket_plan(grp, cams, saturation=False)
        state = G.np32(plan.tile_state).reshape(sc.K, -1)
        _, grads = ov.iteration_plan(sc.partitions(), [c.as_array() for c in cams], plan.view_of_part, sc.sh_degree,
                                     [sc.targets[i] for i in grp], sc.bg, tile_state=state)
        if total is None:
            total = grads
        else:
            for k in range(sc.K):
                for key in scenes.PARAM_KEYS:
                    total[k][key] = total[k][key] + grads[k][key]
    _check_grads(tr, total)


def test_sparse_adam_option(blocks):
    """The visible-only optimiser (an option outside the paper): (1) splx_adam_sparse == splx_adam_groups on the flagged
    rows, bit for bit, and leaves every other row of parameters and moments alone; it clears the flags; (2) the
    flag-driven projection backward stores the first gradient of a row and adds the later ones, never touching the
    rows no view sees; (3) a whole multi-bucket iteration moves exactly the Gaussians some view saw."""
    sc = blocks
    rng = np.random.default_rng(61)
    a, b = _trainer(sc), _trainer(sc)
    n = a.n
    flags = (rng.uniform(size=n) < 0.3)
    g = rng.standard_normal(a.flat["grad"].shape).astype(np.float32)
    m0 = (rng.standard_normal(a.flat["m"].shape) * 0.01).astype(np.float32)
    v0 = (np.abs(rng.standard_normal(a.flat["v"].shape)) * 1e-4).astype(np.float32)
    for tr in (a, b):
        tr.flat["grad"].copy_(torch.from_numpy(g)); tr.flat["m"].copy_(torch.from_numpy(m0)); tr.flat["v"].copy_(torch.from_numpy(v0))
    a.adam_step(n_views=2)                                                   # dense
    touched = torch.from_numpy(flags.astype(np.uint8)).cuda()
    b.ctx.adam_sparse(b.params, b.grads, b.m, b.v, touched, [b.lr[k] for k in scenes.PARAM_KEYS], step=1, grad_scale=0.5)
    torch.cuda.synchronize()
    assert not touched.any()
    fl = torch.from_numpy(flags).cuda()
    for name, init in (("param", None), ("m", m0), ("v", v0)):
        for key in scenes.PARAM_KEYS:
            w = scenes.PARAM_WIDTH[key]
            va = {"param": a.params, "m": a.m, "v": a.v}[name][key].reshape(n, w)
            vb = {"param": b.params, "m": b.m, "v": b.v}[name][key].reshape(n, w)
            assert torch.equal(va[fl], vb[fl]), (name, key)
            orig = torch.from_numpy(np.asarray(sc.params[key], np.float32).reshape(n, w)).cuda() if init is None else None
            if orig is not None:
                assert torch.equal(vb[~fl], orig[~fl]), (name, key)
    # (2) + (3): two iterations over all views with the sparse optimiser
    tr = _trainer(sc)
    tr.sparse_adam = True
    tr.flat["grad"].fill_(float("nan"))                                      # never zeroed, never read where no view looks
    ids = list(range(len(sc.cameras)))
    targets = torch.from_numpy(np.stack(sc.targets)).cuda()
    dense = _trainer(sc)
    dense.lr = {k: 0.0 for k in dense.lr}
    dense.iteration_views(ids, sc.cameras, targets, saturation=False)
    p0 = tr.flat["param"].clone()
    tr.iteration_views(ids, sc.cameras, targets, saturation=False)
    torch.cuda.synchronize()
    assert not tr._touched.any()
    seen = torch.zeros(n, dtype=torch.bool, device="cuda")
    for v_, cam in zip(ids, sc.cameras):
        plan, _ = dense.bucket_plan([v_], [cam], saturation=False)
        dense.forward_plan(plan)
        part = dense.participants(v_, cam)
        vis = dense.proj.radius > 0
        for k in range(sc.K):
            if (part >> k) & 1:
                seen[dense.part_offsets[k]:dense.part_offsets[k + 1]] |= vis[dense.part_offsets[k]:dense.part_offsets[k + 1]]
    assert 0 < int(seen.sum()) < n
    moved = (tr.params["opacity_logit"] != p0[tr._offs["opacity_logit"]:tr._offs["opacity_logit"] + n])
    assert not (moved & ~seen).any()                                         # what no view saw did not move
    assert (moved & seen).float().sum() > 0.9 * seen.float().sum()
    # the gradients of the seen rows are the dense iteration's
    gs = tr.grads["sh"].reshape(n, 48)[seen]; gd = dense.grads["sh"].reshape(n, 48)[seen]
    assert not torch.isnan(gs).any()
    assert float((gs - gd).abs().max()) <= 1e-4 * float(gd.abs().max())


def test_slot_order_is_longest_first_and_changes_nothing(aerial):
    """splx_binning.slot_order: a permutation of the slots with a non-empty list, list lengths descending up to the
    3 % length classes; the blend kernels produce bit-equal partials with and without it, the backward equal gradients."""
    sc = aerial
    cam = sc.cameras[0]
    target = torch.from_numpy(sc.targets[0]).cuda()[None]
    a, b = _trainer(sc), _trainer(sc)
    assert a.bins.slot_order is not None
    b.bins.slot_order = None
    out = []
    for tr in (a, b):
        tr.partials.ct.fill_(float("nan")); tr.partials.d.fill_(float("nan")); tr.partials.n_contrib.fill_(-1)
        plan = tr.make_plan([cam], None, None, True)
        img = tr.forward_plan(plan).clone()
        tr.loss_grad_plan(target)
        tr.backward_plan(overwrite=True)
        torch.cuda.synchronize()
        out.append((img, tr.partials.ct.clone(), tr.partials.d.clone(), tr.partials.n_contrib.clone(), _grads_np(tr)))
    for x, y in zip(out[0][:4], out[1][:4]):
        assert torch.equal(x.view(torch.int32), y.view(torch.int32))
    for key in scenes.PARAM_KEYS:
        assert G.grad_close(out[0][4][key], out[1][4][key]) <= 1e-4, key
    ranges = G.u32(a.bins.tile_ranges).reshape(-1, 2).astype(np.int64)
    length = ranges[:, 1] - ranges[:, 0]
    nslots = length.shape[0]
    order = G.u32(a.bins.slot_order)
    n_live = int(order[nslots])
    assert n_live == int((length > 0).sum())
    assert np.array_equal(np.sort(order[:n_live]), np.nonzero(length > 0)[0])
    ln = length[order[:n_live]].astype(np.float64)
    # descending up to the class width (5 mantissa bits: a later slot is never more than 1/32 longer ... of its binade)
    assert np.all(ln[1:] <= ln[:-1] * (1 + 1 / 16.0) + 1)
    assert ln[0] == length.max()


def _trainer_conservative(sc, **kw):
    tr = G.make_trainer(sc, **kw)
    tr.set_aabbs(*scenes.partition_boxes(sc.params, sc.part_offsets, sub=2))     # sub-cell boxes of means + footprint margin (s21)
    return tr


def test_conservative_regions_change_no_pixel_and_no_gradient(city, blocks):
    """Reading s21: with the boxes of the means grown by splx_footprint_margin the geometric prediction drops no
    non-empty list (device counter num_intersections[1] == 0) and skips no visible Gaussian, so the plan path equals the
    oracle that knows NOTHING of tile states or participants -- images 1e-5 off fragile pixels, gradients 1e-3 -- and
    the all-partition dense GPU path bit for bit."""
    for sc in (city, blocks):
        tr = _trainer_conservative(sc)
        dense = G.make_trainer(sc)
        n_skipped_parts = 0
        for v in (0, len(sc.cameras) - 1):
            cam = sc.cameras[v]
            plan, _ = tr.bucket_plan([v], [cam], saturation=False)
            n_skipped_parts += sum(1 for x in plan.view_of_part if x < 0)
            target = torch.from_numpy(sc.targets[v]).cuda()[None]
            img = tr.iteration_fused(plan, target).clone()
            torch.cuda.synchronize()
            assert int(tr.bins.num_intersections[1].item()) == 0          # no non-empty list dropped as invisible
            res = oracle.iteration(sc.partitions(), cam.as_array(), sc.sh_degree, sc.targets[v], sc.bg)
            frag = _fragile(res)
            ok = G.close(G.np32(img[0]).astype(np.float64), res.image).all(-1)
            assert (~(ok | frag)).sum() == 0
            _check_grads(tr, res.grads, res)
            dense.forward(cam)
            torch.cuda.synchronize()
            assert torch.equal(dense.image, img[0])
        if sc is blocks:
            assert n_skipped_parts > 0          # the prediction does skip whole partitions here


def test_iteration_views_from_host_buffers(blocks):
    """The end-to-end path: splx_iteration with SPLX_ITER_HOST over a multi-bucket iteration -- targets from pinned host
    memory, every image, the loss sums and the intersection counts back to pinned host memory -- equals the same
    iteration on device targets (same kernels; the gradients differ by the atomics' order only)."""
    sc = blocks
    ids = list(range(len(sc.cameras)))
    H, W = sc.cameras[0].height, sc.cameras[0].width
    a, b = _trainer_conservative(sc), _trainer_conservative(sc)
    tg_host = [torch.from_numpy(t).pin_memory() for t in sc.targets]
    img_host = [torch.full((H, W, 3), float("nan")).pin_memory() for _ in ids]
    loss_host = torch.zeros(2, dtype=torch.float64).pin_memory()
    tg_dev = torch.from_numpy(np.stack(sc.targets)).cuda()
    for it in range(2):
        nb = a.iteration_views(ids, sc.cameras, tg_host, saturation=False, images_host=img_host, loss_host=loss_host)
        b.iteration_views(ids, sc.cameras, tg_dev, saturation=False)
        torch.cuda.synchronize()
        assert nb > 1
        tol = 0 if it == 0 else 1e-5
        for v in ids:
            assert torch.allclose(img_host[v].cuda(), b._images[v], rtol=0, atol=tol), (it, v)
            assert torch.equal(img_host[v].cuda(), a._images[v])
        assert float(loss_host[0]) == pytest.approx(float(b.loss_sum[0].item()), rel=1e-6)
        assert float(loss_host[0]) > 0
        a.check_overflow(wait=True)
        assert int(a._m_host[:nb].max()) > 0 and int(a._m_host[:nb].max()) <= a.capacity
    for key in scenes.PARAM_KEYS:
        close = torch.isclose(a.params[key], b.params[key], rtol=1e-3, atol=2e-6)
        assert close.float().mean().item() >= 0.999, key


def test_capacity_overflow_is_reported_by_the_training_path(aerial):
    """a bucket with more intersections than the key capacity must not pass silently: the count comes back
    through splx_iteration's pinned mirror and the trainer raises at its next synchronisation point."""
    from paper_2606_18588_b200.engine import CapacityError
    sc = aerial
    cam = sc.cameras[0]
    full = G.make_trainer(sc)
    full.forward(cam)
    M = full.num_intersections()
    tr = G.make_trainer(sc, capacity=M // 2)
    tg = torch.from_numpy(sc.targets[0]).pin_memory()
    with pytest.raises(CapacityError):
        tr.step_host(0, cam, tg)
    tr2 = _trainer_conservative(sc, capacity=M // 2)
    tr2.iteration_views([0], [cam], torch.from_numpy(sc.targets[0]).cuda()[None], saturation=False)
    with pytest.raises(CapacityError):
        tr2.check_overflow(wait=True)


def test_flag_tracked_gradient_rows_equal_the_plain_buffer(blocks):
    """Trainer.flagged_grads (splx_trainset.touched + splx_adam_groups_flagged): the gradient rows no view reached are
    neither zeroed nor read and count as zero in the DENSE Adam step -- same parameters and moments as the path whose
    first bucket writes every row; gradients equal on the flagged rows; flags == 'some view saw the Gaussian'."""
    sc = blocks
    ids = list(range(len(sc.cameras)))
    targets = torch.from_numpy(np.stack(sc.targets)).cuda()
    a, b = _trainer_conservative(sc), _trainer_conservative(sc)
    a.flagged_grads, b.flagged_grads = True, False
    a._use_flags = lambda plan: True               # (the trainer's own policy would pick the plain pass on a scene this small)
    a.flat["grad"].fill_(float("nan"))             # whatever the untouched rows hold must never be read
    for it in range(3):
        a.iteration_views(ids, sc.cameras, targets, saturation=False)
        b.iteration_views(ids, sc.cameras, targets, saturation=False)
        torch.cuda.synchronize()
    t = a._touched.bool()
    assert 0 < int(t.sum()) < a.n
    for key in scenes.PARAM_KEYS:
        w = scenes.PARAM_WIDTH[key]
        ga, gb = a.grads[key].view(-1, w), b.grads[key].view(-1, w)
        assert torch.isfinite(ga[t]).all()
        assert float((ga[t] - gb[t]).abs().max()) <= 1e-4 * float(gb.abs().max()) + 1e-12, key
        assert not gb[~t].any(), key                                  # the plain path wrote zeros exactly there
        for x, y in ((a.params[key], b.params[key]), (a.m[key], b.m[key]), (a.v[key], b.v[key])):
            assert torch.isfinite(x).all()
            close = torch.isclose(x, y, rtol=1e-3, atol=2e-6)
            assert close.float().mean().item() >= 0.999, key


def test_rows_without_a_2d_gradient_are_skipped_exactly(city):
    """SPLX_PB_SKIP_ZERO: a visible Gaussian that no pixel blended (hidden behind opaque surfaces) has an all-zero 2-D
    gradient row, hence a zero gradient: the flag-tracked projection backward leaves it out like a culled one.  Against
    the run that keeps such rows: the skipped rows are exactly the flagged rows whose gradient is zero there, every other
    flagged row has the same gradient, and the dense Adam steps agree."""
    sc = city
    ids = list(range(len(sc.cameras)))
    targets = torch.from_numpy(np.stack(sc.targets)).cuda()
    a, b = _trainer_conservative(sc), _trainer_conservative(sc)
    b.keep_zero_rows = True
    for tr in (a, b):
        tr._use_flags = lambda plan: True
        tr.flat["grad"].fill_(float("nan"))
    for it in range(2):
        a.iteration_views(ids, sc.cameras, targets, saturation=False)
        b.iteration_views(ids, sc.cameras, targets, saturation=False)
        torch.cuda.synchronize()
    ta, tb = a._touched.bool(), b._touched.bool()
    assert not (ta & ~tb).any()                       # nothing flagged that the keeping run does not flag
    skipped = tb & ~ta
    assert int(skipped.sum()) > 0, "the opaque scene hides no visible Gaussian?"
    for key in scenes.PARAM_KEYS:
        w = scenes.PARAM_WIDTH[key]
        ga, gb = a.grads[key].view(-1, w), b.grads[key].view(-1, w)
        assert not gb[skipped].any(), key             # exactly zero where the row was skipped
        assert torch.isfinite(ga[ta]).all()
        assert float((ga[ta] - gb[ta]).abs().max()) <= 1e-4 * float(gb[tb].abs().max()) + 1e-12, key
        for x, y in ((a.params[key], b.params[key]), (a.m[key], b.m[key]), (a.v[key], b.v[key])):
            close = torch.isclose(x, y, rtol=1e-3, atol=2e-6)
            assert close.float().mean().item() >= 0.999, key


def test_reach_test_on_the_mean_culls_nothing_visible(city, blocks):
    """splx_plan.max_scale: the projection tests a Gaussian's mean against the half spaces outside which nothing of
    that scale reaches the image (reading s21) before it reads scale and rotation.  Same radius / tiles_touched for
    every Gaussian, bit-equal attributes for the visible ones -- and most Gaussians of a view do fail the test."""
    for sc in (city, blocks):
        cam = sc.cameras[-1]
        ms = scenes.partition_boxes(sc.params, sc.part_offsets)[2]
        a, b = G.make_trainer(sc), G.make_trainer(sc)
        pa = binding.Plan([cam], [0] * sc.K, None, True, max_scale=ms)
        pb = binding.Plan([cam], [0] * sc.K, None, True)
        a.ctx.project_plan(a.params, a.part_offsets, pa, a.sh_degree, a.proj)
        b.ctx.project_plan(b.params, b.part_offsets, pb, b.sh_degree, b.proj)
        torch.cuda.synchronize()
        assert torch.equal(a.proj.radius, b.proj.radius) and torch.equal(a.proj.tiles_touched, b.proj.tiles_touched)
        vis = b.proj.radius > 0
        assert 0 < int(vis.sum()) < sc.N
        for name in ("means2d", "depth", "conic_opacity", "rgb", "blend", "clamp"):
            x, y = getattr(a.proj, name), getattr(b.proj, name)
            assert torch.equal(x[vis], y[vis]), name


def _slot_passes(values):
    bits = 1
    while (1 << bits) <= values:
        bits += 1
    return (bits + 7) // 8


def test_renumbered_open_slots_give_the_same_binning(blocks):
    """splx_plan.open_slots (conservative regions: an INVISIBLE slot holds no intersection): the slot sort runs on a
    renumbering of the open slots when that saves a radix pass -- M, keys, vals and ranges bit-equal to the plain plan.
    And a caller whose promise does not hold: the keys that land in an INVISIBLE slot are carried behind every list,
    get no range and are counted in num_intersections[1]; the lists of the open slots are unchanged."""
    sc = blocks
    tr = _trainer_conservative(sc)
    ntiles = tr.bins.tile_ranges.numel() // (2 * tr.K)
    tr._workspaces(sc.cameras[0])
    for v, cam in enumerate(sc.cameras):
        plan, _ = tr.bucket_plan([v], [cam], saturation=False)
        assert plan.open_slots > 0
        nact = sum(1 for k, x in enumerate(plan.view_of_part) if x >= 0 and tr.part_offsets[k + 1] > tr.part_offsets[k])
        saves = _slot_passes(min(plan.open_slots, nact * ntiles) + 1) < _slot_passes(nact * ntiles)
        plain = tr.make_plan(plan.cams, plan.view_of_part, plan.tile_state, True, 0)
        forced = tr.make_plan(plan.cams, plan.view_of_part, plan.tile_state, True, -plan.open_slots)   # even where no pass is saved
        tr.ctx.project_plan(tr.params, tr.part_offsets, plan, tr.sh_degree, tr.proj)
        out = []
        for p in (plain, forced):
            tr.bins.keys.fill_(0); tr.bins.vals.fill_(0)
            launches = tr.ctx.launch_count()
            tr._bin_sort(tr.proj, p, tr.bins, tr._ws_sort)
            M, keys, vals, ranges = G.gpu_bins(tr)
            out.append((M, keys.copy(), vals.copy(), ranges.copy(), int(tr.bins.num_intersections[1]), tr.ctx.launch_count() - launches))
        (M0, k0, v0, r0, d0, l0), (M1, k1, v1, r1, d1, l1) = out
        assert M0 == M1 and M0 > 0 and d0 == 0 and d1 == 0
        assert np.array_equal(k0, k1) and np.array_equal(v0, v1) and np.array_equal(r0, r1)
        assert l1 == l0 - (1 if saves else 0)          # one radix pass less where the renumbering saves one (the map was built with the plan)

    # a broken promise: every second tile of the participating partitions declared INVISIBLE although it holds keys
    v, cam = 0, sc.cameras[0]
    plan, _ = tr.bucket_plan([v], [cam], saturation=False)
    st = plan.tile_state.cpu().numpy().reshape(tr.K, ntiles).copy()
    tr.ctx.project_plan(tr.params, tr.part_offsets, plan, tr.sh_degree, tr.proj)
    tr._bin_sort(tr.proj, tr.make_plan(plan.cams, plan.view_of_part, plan.tile_state, True, 0), tr.bins, tr._ws_sort)
    M0, k0, v0, r0 = [np.copy(x) if isinstance(x, np.ndarray) else x for x in G.gpu_bins(tr)]
    bad = st.copy()
    bad[:, ::2] |= binding.TILE_INVISIBLE
    n_open = int((bad & binding.TILE_INVISIBLE == 0).sum())
    dev = torch.from_numpy(bad.reshape(-1)).cuda()
    tr._bin_sort(tr.proj, tr.make_plan(plan.cams, plan.view_of_part, dev, True, -n_open), tr.bins, tr._ws_sort)
    torch.cuda.synchronize()
    keys = G.u64(tr.bins.keys)[:M0]; vals = G.u32(tr.bins.vals)[:M0]
    ranges = G.u32(tr.bins.tile_ranges).reshape(tr.K, ntiles, 2)
    slot0 = (k0 >> np.uint64(32)).astype(np.int64)
    lost = (bad.reshape(-1)[slot0] & binding.TILE_INVISIBLE) != 0            # keys of the reference that sit in a declared slot
    assert lost.any() and int(tr.bins.num_intersections[1]) == int(lost.sum())
    kept = int((~lost).sum())
    assert np.array_equal(keys[:kept], k0[~lost]) and np.array_equal(vals[:kept], v0[~lost])     # the open lists, in order
    assert ((keys[kept:] >> np.uint64(32)) == tr.K * ntiles + 1).all()
    for k in range(tr.K):
        for t in range(ntiles):
            a, b = r0[k, t]
            if bad[k, t] & binding.TILE_INVISIBLE or a == b:
                assert ranges[k, t, 0] == ranges[k, t, 1] == 0 or ranges[k, t, 0] == ranges[k, t, 1]
            else:
                a1, b1 = ranges[k, t]
                assert b1 - a1 == b - a and np.array_equal(vals[a1:b1], v0[a:b])
