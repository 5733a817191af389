"""-m gpu edge cases of the C ABI: empty inputs and partitions, K = 1, everything culled, capacity
overflow, argument validation.  Expected values come from the oracle or from what the paper's
definitions fix (Eq.5 with no partial = background)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_18588_b200 import binding, scenes
from paper_2606_18588_b200.engine import Trainer
from tests import gpu_common as G

pytestmark = pytest.mark.gpu


def _run_iteration(tr, cam, target):
    tr.forward(cam)
    tr.loss_grad(target)
    tr.backward(overwrite=True)
    torch.cuda.synchronize()


def test_empty_middle_partition_matches_oracle():
    """K = 3 with partition 1 empty: its partial is the identity (0,0,0,T=1) everywhere."""
    sc = scenes.tiny(n=1500, size=64, f=75.0, K=2, seed=5)
    a = int(sc.part_offsets[1])
    offs = np.array([0, a, a, sc.N], np.int64)
    cam = sc.cameras[0]
    tr = Trainer(sc.params, offs, cam.width, cam.height, sc.sh_degree, sc.bg)
    target = torch.from_numpy(sc.targets[0]).cuda()
    _run_iteration(tr, cam, target)
    ct = G.np32(tr.partials.ct)
    assert not ct[1, ..., :3].any() and (ct[1, ..., 3] == 1).all()
    assert not G.u32(tr.partials.n_contrib)[1].any()
    parts = [sc.partition(0), {k: v[:0] for k, v in sc.partition(0).items()}, sc.partition(1)]
    res = oracle.iteration(parts, cam.as_array(), sc.sh_degree, sc.targets[0], sc.bg)
    frag = np.zeros((cam.height, cam.width), bool)
    for pa in res.partials:
        frag |= pa.margin < G.FRAGILE_MARGIN
    ok = G.close(G.np32(tr.image), res.image).all(-1)
    assert (ok | frag).all()
    for key in scenes.PARAM_KEYS:
        ref = np.concatenate([g[key].reshape(-1) for g in res.grads])
        assert G.rel_l2(G.np32(tr.grads[key]), ref) <= 1e-3, key


def test_zero_gaussians_gives_background():
    """n = 0: Eq.5 with no partial -> image = bg, T_total = 1; nothing is launched that could fault."""
    sc = scenes.tiny(n=64, size=48, f=60.0, K=2, seed=6)
    empty = {k: v[:0] for k, v in sc.params.items()}
    cam = sc.cameras[0]
    bg = (0.25, 0.5, 0.75)
    tr = Trainer(empty, np.zeros(3, np.int64), cam.width, cam.height, sc.sh_degree, bg)
    _run_iteration(tr, cam, torch.from_numpy(sc.targets[0]).cuda())
    assert tr.num_intersections() == 0
    img = G.np32(tr.image)
    assert np.allclose(img, np.asarray(bg, np.float32)[None, None, :], atol=0)
    assert (G.np32(tr.T_total) == 1).all()


def test_all_gaussians_behind_the_camera():
    sc = scenes.tiny(n=512, size=48, f=60.0, K=2, seed=7)
    sc.params["mean"][:, 2] *= -1.0          # z <= near: culled by the mean
    cam = sc.cameras[0]
    tr = Trainer(sc.params, sc.part_offsets, cam.width, cam.height, sc.sh_degree, sc.bg)
    _run_iteration(tr, cam, torch.from_numpy(sc.targets[0]).cuda())
    assert tr.num_intersections() == 0
    assert not G.np32(tr.proj.radius).any() and not G.np32(tr.image).any()
    for key in scenes.PARAM_KEYS:
        assert not G.np32(tr.grads[key]).any(), key     # overwrite mode writes zeros for culled rows


def test_k1_is_partial_plus_background():
    """north_star check 1: K = 1 composition equals the direct render (+ T*bg)."""
    sc = scenes.tiny(n=2000, size=80, f=90.0, K=1, seed=8)
    cam = sc.cameras[0]
    bg = (0.1, 0.2, 0.3)
    tr = Trainer(sc.params, sc.part_offsets, cam.width, cam.height, sc.sh_degree, bg)
    tr.forward(cam)
    torch.cuda.synchronize()
    ct = G.np32(tr.partials.ct)[0].astype(np.float64)
    expect = ct[..., :3] + ct[..., 3:4] * np.asarray(bg)
    assert np.abs(G.np32(tr.image) - expect).max() <= 1e-6
    assert np.array_equal(G.np32(tr.T_total), G.np32(tr.partials.ct)[0][..., 3])


def test_capacity_overflow_is_reported_and_harmless():
    sc = scenes.tiny(n=4096, size=128, K=2)
    cam = sc.cameras[0]
    full = Trainer(sc.params, sc.part_offsets, cam.width, cam.height, sc.sh_degree, sc.bg)
    full.forward(cam)
    M = full.num_intersections()
    small = Trainer(sc.params, sc.part_offsets, cam.width, cam.height, sc.sh_degree, sc.bg, capacity=M // 2)
    small.forward(cam)                       # must not write out of bounds or hang
    with pytest.raises(binding.SplxError) as e:
        small.num_intersections()
    assert e.value.code == binding.ERR_CAPACITY and str(M) in str(e.value)
    exact = Trainer(sc.params, sc.part_offsets, cam.width, cam.height, sc.sh_degree, sc.bg, capacity=M)
    exact.forward(cam)
    assert exact.num_intersections() == M
    assert torch.equal(exact.image, full.image)


def test_argument_validation():
    sc = scenes.tiny(n=128, size=32, f=40.0, K=2, seed=9)
    cam = sc.cameras[0]
    tr = Trainer(sc.params, sc.part_offsets, cam.width, cam.height, sc.sh_degree, sc.bg)
    tr._workspaces(cam)
    with pytest.raises(binding.SplxError) as e:
        tr.ctx.project(tr.params, cam, 4, tr.proj)
    assert e.value.code == binding.ERR_INVALID_ARG
    with pytest.raises(binding.SplxError) as e:
        tr.ctx.bin_sort(tr.proj, 2, [0, 5, 3], cam, tr.bins, tr._ws_sort)       # not monotone / not ending at n
    assert e.value.code == binding.ERR_INVALID_ARG
    with pytest.raises(binding.SplxError) as e:
        tr.ctx.bin_sort(tr.proj, 2, tr.part_offsets, cam, tr.bins, tr._ws_sort[:64])
    assert e.value.code == binding.ERR_WORKSPACE
    p = torch.zeros(16, device="cuda")
    with pytest.raises(binding.SplxError):
        tr.ctx.adam(p, p.clone(), p.clone(), p.clone(), lr=1e-3, step=0)         # step is 1-based


# ---- the same edges under launch plans ------------------------------------------------------------------
def test_plan_without_participants_gives_background():
    """Every partition at view -1: nothing is projected, binned or rendered; Eq.5 with no partial = background for
    every view; '=' mode writes an all-zero gradient."""
    sc = scenes.tiny(n=600, size=48, f=60.0, K=2, seed=7)
    cam = sc.cameras[0]
    bg = (0.1, 0.2, 0.3)
    tr = Trainer(sc.params, sc.part_offsets, cam.width, cam.height, sc.sh_degree, bg)
    for v in tr.grads.values():
        v.fill_(3.0)
    plan = tr.make_plan([cam, cam], [-1, -1], None, True)
    target = torch.from_numpy(np.stack([sc.targets[0], sc.targets[0]])).cuda()
    imgs = tr.iteration_fused(plan, target, overwrite=True)
    torch.cuda.synchronize()
    assert tr.num_intersections() == 0
    assert np.allclose(G.np32(imgs), np.asarray(bg, np.float32), atol=0)
    assert (G.np32(tr._T_totals[:2]) == 1).all()
    assert not tr.flat["grad"].any()


def test_plan_with_64_partitions_and_8_views():
    """The limits of the plan: K = SPLX_MAX_K = 64 partitions, B = SPLX_MAX_VIEWS = 8 views (each rendering 8 of
    them), against the oracle's plan iteration."""
    sc = scenes.tiny(n=3200, size=64, f=75.0, K=64, seed=8, sh_degree=1)
    base = sc.cameras[0]
    cams = []
    for b in range(8):
        t = base.t + np.array([0.05 * b, -0.03 * b, 0.1 * b], np.float32)
        cams.append(scenes.Camera(base.R, t, base.fx, base.fy, base.cx, base.cy, base.width, base.height))
    vop = [k % 8 for k in range(64)]
    rng = np.random.default_rng(9)
    targets = rng.uniform(0, 1, (8, 64, 64, 3)).astype(np.float32)
    tr = Trainer(sc.params, sc.part_offsets, 64, 64, sc.sh_degree, sc.bg)
    plan = tr.make_plan(cams, vop, None, True)
    imgs = tr.iteration_fused(plan, torch.from_numpy(targets).cuda(), overwrite=True).clone()
    torch.cuda.synchronize()
    from oracle import visibility as ov
    views, grads = ov.iteration_plan(sc.partitions(), [c.as_array() for c in cams], vop, sc.sh_degree, list(targets), sc.bg)
    for b, res in enumerate(views):
        frag = np.zeros((64, 64), bool)
        for pa in res.partials:
            frag |= pa.margin < G.FRAGILE_MARGIN
        frag |= res.order_margin < 1e-6
        ok = G.close(G.np32(imgs[b]).astype(np.float64), res.image).all(-1)
        assert (ok | frag).all(), b
    for key in scenes.PARAM_KEYS:
        ref = np.concatenate([g[key].reshape(-1) for g in grads])
        assert G.rel_l2(G.np32(tr.grads[key]), ref) <= 1e-3, key


def test_plan_capacity_overflow_and_bad_plans_are_reported():
    sc = scenes.tiny(n=2000, size=64, f=75.0, K=2, seed=10)
    cam = sc.cameras[0]
    tr = Trainer(sc.params, sc.part_offsets, cam.width, cam.height, sc.sh_degree, sc.bg, capacity=1000)
    plan = tr.make_plan([cam], [0, 0], None, True)
    tr.forward_plan(plan)
    with pytest.raises(binding.SplxError) as e:
        tr.num_intersections()
    assert e.value.code == binding.ERR_CAPACITY
    other = scenes.Camera(cam.R, cam.t, cam.fx, cam.fy, cam.cx, cam.cy, cam.width * 2, cam.height)
    for bad in (lambda: tr.make_plan([cam, other], [0, 1]),          # views of different sizes
                lambda: tr.make_plan([cam], [0, 1]),                 # view index out of range
                lambda: tr.make_plan([cam] * 9, [0, 0])):            # more than SPLX_MAX_VIEWS views
        with pytest.raises(binding.SplxError) as e:
            tr.ctx.project_plan(tr.params, tr.part_offsets, bad(), tr.sh_degree, tr.proj)
        assert e.value.code == binding.ERR_INVALID_ARG
    with pytest.raises(binding.SplxError):                            # sparse compose without the binning
        tr.ctx.compose_plan(tr.partials, None, plan, tr.bg, tr._images[:1])


def test_cross_boundary_argument_errors_and_degenerate_inputs():
    """splx_cross_sets / splx_bin_sort_filtered_plan: invalid boxes and K are refused; one partition has no Q_cross;
    a NULL mask is the unfiltered binning."""
    import numpy as np
    from paper_2606_18588_b200 import binding, scenes
    sc = scenes.small_aerial(n=3000)
    tr = G.make_trainer(sc)
    lo, hi = scenes.partition_aabbs(sc.params, sc.part_offsets, inflate_sigma=0.0)
    mask = torch.empty(tr.n, dtype=torch.int64, device="cuda")
    bad_hi = hi.copy(); bad_hi[1, 0] = lo[1, 0] - 1.0
    with pytest.raises(binding.SplxError):
        tr.ctx.cross_sets(tr.params, tr.part_offsets, lo, bad_hi, mask)
    with pytest.raises(binding.SplxError):
        tr.ctx.cross_sets(tr.params, tr.part_offsets, lo, hi, mask, support_sigma=-1.0)
    with pytest.raises(binding.SplxError):
        tr.ctx.cross_sets(tr.params, tr.part_offsets, lo[:2], hi[:2], mask)      # K does not match part_offsets
    # a single partition: nothing to cross into
    one = np.array([0, tr.n], np.int64)
    tr.ctx.cross_sets(tr.params, one, lo.min(0, keepdims=True), hi.max(0, keepdims=True), mask)
    torch.cuda.synchronize()
    assert not mask.any()
    # NULL mask == splx_bin_sort_plan
    cam = sc.cameras[0]
    plan = tr.make_plan([cam], None, None, False)
    tr._workspaces(cam)
    tr.ctx.project_plan(tr.params, tr.part_offsets, plan, tr.sh_degree, tr.proj)
    tr.ctx.bin_sort_plan(tr.proj, tr.part_offsets, plan, tr.bins, tr._ws_sort)
    M0, k0, v0, r0 = G.gpu_bins(tr)
    k0, v0, r0 = k0.copy(), v0.copy(), r0.copy()
    tr.ctx.bin_sort_filtered_plan(tr.proj, tr.part_offsets, plan, None, np.zeros((tr.K, 2), np.float32), tr.bins, tr._ws_sort)
    M1, k1, v1, r1 = G.gpu_bins(tr)
    assert M1 == M0 and np.array_equal(k1, k0) and np.array_equal(v1, v0) and np.array_equal(r1, r0)
