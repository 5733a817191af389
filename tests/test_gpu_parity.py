"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by
element, on seeded inputs.  Stage-wise and teacher-forced (each oracle stage is fed the GPU's
previous-stage output) for the bit-exact integer work; free-running end to end for the floats.
Bars (BASELINE.json north_star): bit-exact intersection counts / sorted keys / tile ranges;
1e-5 abs/rel on images and T; 1e-3 rel on accumulated gradients."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_18588_b200 import scenes
from tests import gpu_common as G

pytestmark = pytest.mark.gpu

def _big_footprints():
    """Footprints of ~20-60 tiles (mean > 16): takes the load-balanced key emission (k_emit_keys_lb) of street-level views."""
    sc = scenes.tiny(n=700, size=176, f=200.0, K=3, sh_degree=1, seed=4)
    sc.params["log_scale"] = (sc.params["log_scale"] + 1.6).astype(np.float32)
    sc.params["opacity_logit"] = (sc.params["opacity_logit"] - 2.0).astype(np.float32)
    sc.name = "tiny_big_footprints"
    return sc


SCENES = {
    "tiny": lambda: scenes.tiny(),                              # BASELINE configs[0]
    "aerial_small": lambda: scenes.small_aerial(),              # configs[1] recipe, ragged 320x176, K=4, SH3
    "tiny_k5_sh2": lambda: scenes.tiny(n=3000, size=72, f=84.0, K=5, sh_degree=2, seed=3),  # ragged both ways
    "big_footprints": _big_footprints,
}


class Run:
    """One GPU iteration, stage by stage, with every intermediate copied to the host."""

    def __init__(self, sc):
        self.sc = sc
        self.cam = sc.cameras[0]
        self.camv = self.cam.as_array()
        self.W, self.H = self.cam.width, self.cam.height
        tr = self.tr = G.make_trainer(sc)
        c = tr.ctx
        tr._workspaces(self.cam); tr._cam = self.cam
        c.project(tr.params, self.cam, tr.sh_degree, tr.proj)
        self.proj = G.gpu_projected(tr)
        c.bin_sort(tr.proj, tr.K, tr.part_offsets, self.cam, tr.bins, tr._ws_sort)
        self.M, self.keys, self.vals, self.ranges = G.gpu_bins(tr)
        c.render_partial(tr.proj, tr.bins, tr.K, self.cam, tr.partials, tr.pairs)
        self.ct = G.np32(tr.partials.ct).astype(np.float64)
        self.d = G.np32(tr.partials.d).astype(np.float64)
        self.n_contrib = G.u32(tr.partials.n_contrib)
        self.pairs = int(tr.pairs[0].item()); self.blended = int(tr.pairs[1].item())
        c.compose(tr.K, tr.partials, self.cam, tr.bg, tr.image, tr.T_total)
        self.image = G.np32(tr.image).astype(np.float64)
        self.T_total = G.np32(tr.T_total).astype(np.float64)
        self.target = torch.from_numpy(sc.targets[0]).cuda()
        tr.loss_sum.zero_()
        c.l1_loss_grad(tr.image, self.target, tr.g_image, tr.loss_sum)
        self.g_image = G.np32(tr.g_image).astype(np.float64)
        self.loss = float(tr.loss_sum[0].item()) / self.g_image.size
        torch.cuda.synchronize()


_cache = {}


@pytest.fixture(params=list(SCENES))
def run(request):
    if request.param not in _cache:
        _cache[request.param] = Run(SCENES[request.param]())
    return _cache[request.param]


def _oracle_partition_bins(run, k):
    a, b = run.tr.part_offsets[k], run.tr.part_offsets[k + 1]
    pr = run.proj
    return oracle.bin_sort(pr.means2d[a:b], pr.radius[a:b], pr.depth[a:b], run.W, run.H)


def test_a1_projection(run):
    sc, pr = run.sc, run.proj
    ref = oracle.project(sc.params["mean"], sc.params["log_scale"], sc.params["quat"], sc.params["opacity_logit"],
                         sc.params["sh"], sc.sh_degree, run.camv)
    # integer decision radius = ceil(3 sqrt(lambda)): equal unless 3 sqrt(lambda) is within 1e-5 of an integer
    r3 = np.where(ref.radius > 0, ref.radius / (1.0 + np.where(np.isfinite(ref.radius_margin), ref.radius_margin, 0)), 1.0)
    near_int = np.minimum(ref.radius - r3, r3 - (ref.radius - 1)) / r3 < 1e-5
    vis_ref, vis = ref.radius > 0, pr.radius > 0
    agree = vis_ref & vis & (ref.radius == pr.radius)
    bad_radius = (vis_ref & vis & (ref.radius != pr.radius) & ~near_int).sum()
    assert bad_radius == 0
    # culling may differ only through a radius flip or a tile-rect flip at a tile boundary (rare)
    assert (vis_ref != vis).sum() <= max(2, 1e-4 * len(vis))
    assert agree.sum() >= 0.999 * vis_ref.sum()
    m = agree
    # 2-D mean: u = fx x/z + cx is stored in fp32 at image scale, so its absolute error is a few
    # ulp(max(W,H)) whatever |u| is: 4 * 2^-23 * max(W,H) px
    ulp_img = 4 * 2.0 ** -23 * max(run.W, run.H)
    assert (G.close(pr.means2d[m], ref.means2d[m]) | (np.abs(pr.means2d[m] - ref.means2d[m]) <= ulp_img)).all()
    assert G.close(pr.depth[m], ref.depth[m]).all()
    # the depth is the sort key: both sides evaluate it in fp32 in one fixed operation order (reading s12) -- bit-equal
    dk = oracle.depth_key(sc.params["mean"], run.camv)
    assert np.array_equal(pr.depth[m].astype(np.float32).view(np.uint32), dk[m].astype(np.float32).view(np.uint32))
    assert G.close(pr.rgb[m], ref.rgb[m]).all()
    assert G.close(pr.conic_opacity[m, 3], ref.conic_opacity[m, 3]).all()
    # conic = Sigma2D^-1: relative error amplified by the conditioning a*c/det of the 2x2 inverse
    # (DESIGN.md 'Tolerances'): allow 1e-5 * max(1, kappa/4)
    A, B, Cc = ref.conic_opacity[m, 0], ref.conic_opacity[m, 1], ref.conic_opacity[m, 2]
    kappa = (A * Cc) / (A * Cc - B * B)
    scale = np.maximum(np.maximum(np.abs(A), np.abs(Cc)), 1.0)
    err = np.abs(pr.conic_opacity[m, :3] - ref.conic_opacity[m, :3]).max(1)
    assert (err <= 1e-5 * scale * np.maximum(1.0, kappa / 4)).all()
    assert (err <= 1e-5 * scale).mean() > 0.99
    assert (pr.clamp[m] != ref.clamp[m]).sum() <= 2   # a colour channel within rounding of 0
    # culled Gaussians: radius 0 and no tiles (their other attributes are not written)
    assert not pr.radius[~vis].any() and not pr.tiles_touched[~vis].any()


def test_a2_a4_binning_bit_exact(run):
    pr = run.proj
    if run.sc.name == "tiny_big_footprints":
        assert run.M > 16 * (pr.radius > 0).sum(), "this scene must take the load-balanced emission path"
    # teacher-forced: counts from the GPU's own (means2d, radius)
    M_ref, tt_ref = oracle.count_tiles(pr.means2d, pr.radius, run.W, run.H)
    assert np.array_equal(pr.tiles_touched, tt_ref)
    assert run.M == M_ref
    ntiles = run.ranges.shape[1]
    pos = 0
    for k in range(run.tr.K):
        b = _oracle_partition_bins(run, k)
        seg_keys = run.keys[pos:pos + b.M]
        seg_vals = run.vals[pos:pos + b.M]
        assert np.array_equal(seg_keys >> np.uint64(32), (b.keys >> np.uint64(32)) + np.uint64(k * ntiles))
        assert np.array_equal(seg_keys & np.uint64(0xFFFFFFFF), b.keys & np.uint64(0xFFFFFFFF))
        assert np.array_equal(seg_vals, b.vals + np.uint32(run.tr.part_offsets[k]))
        live = b.ranges[:, 1] > b.ranges[:, 0]
        assert np.array_equal(run.ranges[k][live], b.ranges[live] + np.uint32(pos))
        assert not run.ranges[k][~live].any()
        pos += b.M
    assert pos == run.M


def _oracle_partials(run):
    pr = run.proj
    out = []
    pos = 0
    for k in range(run.tr.K):
        a, b = run.tr.part_offsets[k], run.tr.part_offsets[k + 1]
        bins = _oracle_partition_bins(run, k)
        out.append((oracle.render_partial(pr.means2d[a:b], pr.conic_opacity[a:b], pr.rgb[a:b], pr.depth[a:b],
                                          bins.vals, bins.ranges, run.W, run.H), bins))
    return out


def test_a5_local_render(run):
    refs = _oracle_partials(run)
    walked = 0
    n_frag = 0
    for k, (ref, _) in enumerate(refs):
        walked += ref.walked
        frag = ref.margin < G.FRAGILE_MARGIN
        n_frag += int(frag.sum())
        ok_ct = G.close(run.ct[k], ref.ct).all(-1)
        ok_d = G.close(run.d[k], ref.d)
        assert (ok_ct | frag).all(), f"partition {k}: {(~(ok_ct | frag)).sum()} robust pixels off"
        assert (ok_d | frag).all()
        assert ((run.n_contrib[k] == ref.n_contrib) | frag).all()
        # fragile pixels: a flipped decision moves the pixel by a bounded amount
        assert (np.abs(run.ct[k] - ref.ct).max(-1) <= G.FRAGILE_TOL)[frag].all()
        T = run.ct[k][..., 3]
        assert (T <= 1).all() and (T >= 1e-4 * (1 - 1e-5)).all()
    assert n_frag <= 2e-3 * run.tr.K * run.W * run.H
    # unit of work counted by the kernel == the oracle's, up to fragile early-exit positions
    assert abs(run.pairs - walked) <= 1e-3 * walked + 64
    blended_ref = 0
    for k, (ref, bins) in enumerate(refs):
        # contributors of a pixel = entries of its list that were blended; recount with the oracle's weights:
        # sum_i alpha_i T_i = 1 - T  holds per pixel, the count itself comes from a second oracle walk
        blended_ref += int((ref.ct[..., 3] < 1).sum())
    assert run.blended >= blended_ref   # at least one blended pair per non-empty pixel


def test_a6_composition(run):
    img, Tt, order, om = oracle.compose(run.ct, run.d, run.tr.bg)
    robust = ~(om < 1e-6)
    ok = G.close(run.image, img).all(-1) & G.close(run.T_total, Tt)
    assert (ok | ~robust).all()
    # order-fragile pixels (two ordering keys within fp32 rounding): accept the swapped order
    assert (~robust).sum() <= 1e-3 * run.W * run.H
    assert np.abs(run.image - img).max() <= 1e-2


def test_a7_loss(run):
    L, g = oracle.l1(run.image, run.sc.targets[0])
    assert run.loss == pytest.approx(L, rel=1e-5)
    assert np.array_equal(run.g_image.astype(np.float32), g.astype(np.float32))


def test_a8_composition_backward(run):
    tr = run.tr
    rng = np.random.default_rng(7)
    gT = rng.standard_normal((run.H, run.W)).astype(np.float32)
    g_ct = torch.empty((tr.K, run.H, run.W, 4), dtype=torch.float32, device="cuda")
    tr.ctx.compose_backward(tr.K, tr.partials, run.cam, tr.bg, tr.g_image, torch.from_numpy(gT).cuda(), g_ct)
    got = G.np32(g_ct).astype(np.float64)
    ref = oracle.compose_bwd(run.ct, run.d, run.g_image, tr.bg, gT)
    _, _, _, om = oracle.compose(run.ct, run.d, tr.bg)
    robust = ~(om < 1e-6)
    scale = np.abs(ref).max()
    assert (np.abs(got - ref)[:, robust] <= 1e-5 * scale).all()


def test_a9_raster_backward(run):
    tr = run.tr
    refs = _oracle_partials(run)
    rng = np.random.default_rng(8)
    g_ct = rng.standard_normal((tr.K, run.H, run.W, 4)).astype(np.float32)
    for k, (ref, _) in enumerate(refs):
        g_ct[k][ref.margin < G.FRAGILE_MARGIN] = 0   # fragile pixels take no part (both sides)
    g2d = torch.zeros((tr.n, 12), dtype=torch.float32, device="cuda")
    tr.ctx.raster_backward(tr.proj, tr.bins, tr.K, run.cam, tr.partials, torch.from_numpy(g_ct).cuda(), g2d)
    got = G.np32(g2d).astype(np.float64)
    g2d2 = torch.zeros_like(g2d)
    tr.ctx.raster_backward(tr.proj, tr.bins, tr.K, run.cam, tr.partials, torch.from_numpy(g_ct).cuda(), g2d2)
    got2 = G.np32(g2d2).astype(np.float64)
    assert not got[:, 9:].any()
    pr = run.proj
    ref_all = np.zeros((tr.n, 9))
    for k, (_, bins) in enumerate(refs):
        a, b = tr.part_offsets[k], tr.part_offsets[k + 1]
        gm, gc, go, gr = oracle.raster_bwd(pr.means2d[a:b], pr.conic_opacity[a:b], pr.rgb[a:b], bins.vals,
                                           bins.ranges, run.W, run.H, g_ct[k])
        ref_all[a:b] = np.concatenate([gm, gc, go[:, None], gr], 1)
    for name, sl in (("means2d", slice(0, 2)), ("conic", slice(2, 5)), ("opacity", slice(5, 6)), ("rgb", slice(6, 9))):
        assert G.grad_close(got[:, sl], ref_all[:, sl]) <= 1e-3, name
        assert G.rel_l2(got[:, sl], ref_all[:, sl]) <= 1e-3, name
        # atomic-order noise between two runs is far below the bar
        assert G.grad_close(got2[:, sl], got[:, sl]) <= 1e-4, name
    assert np.abs(ref_all).max() > 0


def test_a10_projection_backward(run):
    tr, sc = run.tr, run.sc
    rng = np.random.default_rng(9)
    g2d = np.zeros((tr.n, 12), np.float32)
    g2d[:, :9] = rng.standard_normal((tr.n, 9)) * np.array([1, 1, 5, 5, 5, 1, 1, 1, 1])
    grads = {k: torch.zeros_like(v) for k, v in tr.params.items()}
    g2d_dev = torch.from_numpy(g2d).cuda()
    tr.ctx.project_backward(tr.params, run.cam, tr.sh_degree, tr.proj, g2d_dev, grads, clear_g2d=True)
    pr = run.proj
    ref = oracle.project_bwd(sc.params["mean"], sc.params["log_scale"], sc.params["quat"], sc.params["opacity_logit"],
                             sc.params["sh"], sc.sh_degree, run.camv, pr.radius, pr.clamp, g2d[:, 0:2], g2d[:, 2:5],
                             g2d[:, 5], g2d[:, 6:9])
    for key in scenes.PARAM_KEYS:
        got = G.np32(grads[key]).reshape(ref[key].shape)
        assert G.grad_close(got, ref[key]) <= 1e-3, key
        assert G.rel_l2(got, ref[key]) <= 1e-4, key
    vis = pr.radius > 0
    assert not G.np32(g2d_dev)[vis].any() and np.array_equal(G.np32(g2d_dev)[~vis], g2d[~vis])
    # accumulation (+=): a second call doubles the gradient
    g2d_dev = torch.from_numpy(g2d).cuda()
    before = grads["mean"].clone()
    tr.ctx.project_backward(tr.params, run.cam, tr.sh_degree, tr.proj, g2d_dev, grads)
    assert torch.allclose(grads["mean"], 2 * before, rtol=1e-6, atol=0)
    # overwrite mode (=): every row written, whatever the buffers held before; equals the += result from zero
    dirty = {k: torch.full_like(v, 123.0) for k, v in tr.params.items()}
    g2d_dev = torch.from_numpy(g2d).cuda()
    tr.ctx.project_backward(tr.params, run.cam, tr.sh_degree, tr.proj, g2d_dev, dirty, overwrite=True)
    clean = {k: torch.zeros_like(v) for k, v in tr.params.items()}
    g2d_dev = torch.from_numpy(g2d).cuda()
    tr.ctx.project_backward(tr.params, run.cam, tr.sh_degree, tr.proj, g2d_dev, clean)
    for key in scenes.PARAM_KEYS:
        assert torch.equal(dirty[key], clean[key]), key


def test_free_running_iteration_end_to_end(run):
    """The whole path free-running on both sides: image/T at 1e-5 (robust pixels), gradients at 1e-3."""
    tr, sc = run.tr, run.sc
    res = oracle.iteration(sc.partitions(), run.camv, sc.sh_degree, sc.targets[0], sc.bg)
    frag = np.zeros((run.H, run.W), bool)
    for pa in res.partials:
        frag |= pa.margin < G.FRAGILE_MARGIN
    frag |= res.order_margin < 1e-6
    # Gaussians whose radius decision differs change which tiles list them: exclude their pixels via the image check
    ok = G.close(run.image, res.image).all(-1) & G.close(run.T_total, res.T_total)
    n_bad = (~(ok | frag)).sum()
    assert n_bad <= 1e-4 * run.W * run.H, f"{n_bad} robust pixels differ by more than 1e-5"
    assert frag.sum() <= 4e-3 * run.W * run.H
    assert run.loss == pytest.approx(res.loss, rel=1e-5)
    tr.zero_grad()
    tr.backward()
    G.check_grads(tr, res.grads, res)


def test_a11_adam(run):
    tr = run.tr
    rng = np.random.default_rng(11)
    n = 100_003   # not a multiple of 4: exercises the scalar tail
    p0 = rng.standard_normal(n).astype(np.float32)
    p = torch.from_numpy(p0.copy()).cuda(); m = torch.zeros_like(p); v = torch.zeros_like(p)
    P = p0.astype(np.float64); Mo = np.zeros(n); Vo = np.zeros(n)
    # aligned views (tail included) from one allocation
    for step in range(1, 6):
        g = (rng.standard_normal(n) * 10.0 ** rng.uniform(-4, 1, n)).astype(np.float32)
        gd = torch.from_numpy(g.copy()).cuda()
        tr.ctx.adam(p, gd, m, v, lr=3e-3, step=step, grad_scale=0.5, zero_grad=True)
        oracle.adam(P, g.astype(np.float64) * 0.5, Mo, Vo, lr=float(np.float32(3e-3)), beta1=float(np.float32(0.9)),
                    beta2=float(np.float32(0.999)), eps=float(np.float32(1e-15)), step=step)
        assert not gd.any()
    assert np.abs(G.np32(p) - P).max() <= 1e-5
    assert G.rel_l2(G.np32(m), Mo) <= 1e-5 and G.rel_l2(G.np32(v), Vo) <= 1e-5


def test_a11_adam_groups_equals_per_group_calls(run):
    """splx_adam_groups (one launch over the flat buffer) == one splx_adam call per group, bit for bit."""
    tr = run.tr
    rng = np.random.default_rng(12)
    offs = [0, 1000, 1000, 5004, 9008]      # an empty group included; multiples of 4
    lrs = [1e-3, 7e-2, 3e-4, 5e-3]
    n = offs[-1]
    p0 = rng.standard_normal(n).astype(np.float32)
    g0 = rng.standard_normal(n).astype(np.float32)
    a = [torch.from_numpy(x.copy()).cuda() for x in (p0, g0, np.zeros(n, np.float32), np.zeros(n, np.float32))]
    b = [t.clone() for t in a]
    for step in (1, 2, 3):
        tr.ctx.adam_groups(a[0], a[1], a[2], a[3], offs, lrs, step=step, grad_scale=0.25)
        for j, lr in enumerate(lrs):
            s = slice(offs[j], offs[j + 1])
            if offs[j + 1] > offs[j]:
                tr.ctx.adam(b[0][s], b[1][s], b[2][s], b[3][s], lr=lr, step=step, grad_scale=0.25)
    for x, y in zip(a, b):
        assert torch.equal(x, y)
    # and against the oracle
    P = p0.astype(np.float64); Mo = np.zeros(n); Vo = np.zeros(n)
    for step in (1, 2, 3):
        for j, lr in enumerate(lrs):
            s = slice(offs[j], offs[j + 1])
            Ps, Ms, Vs = P[s].copy(), Mo[s].copy(), Vo[s].copy()
            oracle.adam(Ps, g0[s].astype(np.float64) * 0.25, Ms, Vs, lr=float(np.float32(lr)), beta1=float(np.float32(0.9)),
                        beta2=float(np.float32(0.999)), eps=float(np.float32(1e-15)), step=step)
            P[s], Mo[s], Vo[s] = Ps, Ms, Vs
    assert np.abs(G.np32(a[0]) - P).max() <= 1e-5
