"""-m gpu parity of the loss of PAPER.md L95, L = L_RGB + lambda L_D-SSIM (reading s33), through the C ABI
(splx_dssim_loss_grad, and splx_iteration with lambda_dssim > 0) against oracle/dssim.py.
Bars: the loss at 1e-5, dL/dimage and the accumulated parameter gradients at 1e-3 (north_star)."""
import numpy as np
import pytest
import torch

import oracle
from oracle import dssim as od
from paper_2606_18588_b200 import binding, scenes
from tests import gpu_common as G

pytestmark = pytest.mark.gpu


def _cam(W, H):
    return scenes.Camera(np.eye(3, dtype=np.float32), np.zeros(3, np.float32), 50.0, 50.0, W / 2, H / 2, W, H)


def _run(ctx, x, y, lam):
    """x, y: numpy [B,H,W,3] float32.  Returns (loss sums [2], dL/dimage)."""
    B, H, W, _ = x.shape
    cam = _cam(W, H)
    xd, yd = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
    g = torch.full_like(xd, float("nan"))
    ls = torch.zeros(2, dtype=torch.float64, device="cuda")
    ws = torch.empty(B * ctx.dssim_ws_floats(W, H), dtype=torch.float32, device="cuda")
    ctx.dssim_loss_grad(cam, xd, yd, g, ls, ws, lam)
    torch.cuda.synchronize()
    return ls.cpu().numpy(), g.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("shape", [(1, 53, 70), (2, 16, 16), (3, 40, 37), (1, 7, 5)])     # ragged tiles, several views, smaller than the window
def test_dssim_loss_and_gradient_against_the_oracle(shape):
    B, H, W = shape
    rng = np.random.default_rng(B * 1000 + H)
    x = rng.uniform(0, 1, (B, H, W, 3)).astype(np.float32)
    y = (0.6 * x + 0.4 * rng.uniform(0, 1, (B, H, W, 3))).astype(np.float32)       # correlated: SSIM well away from 0
    lam = 0.2
    ctx = binding.Context(0)
    ls, g = _run(ctx, x, y, lam)
    count = H * W * 3
    l1_ref = ssim_ref = 0.0
    for b in range(B):
        L, l1, m, gref = od.loss(x[b], y[b], lam)
        l1_ref += l1; ssim_ref += m
        assert G.grad_close(g[b], gref) <= 1e-3 and G.rel_l2(g[b], gref) <= 1e-3, b
        # per element, not only against the tensor maximum: |err| <= 1e-3 |ref| + 1e-4 max|ref|
        assert (np.abs(g[b] - gref) <= 1e-3 * np.abs(gref) + 1e-4 * np.abs(gref).max()).all(), b
    assert ls[0] / count == pytest.approx(l1_ref, rel=1e-5)
    assert ls[1] / count == pytest.approx(ssim_ref, abs=1e-5 * B)


def test_identical_images_and_lambda_zero():
    rng = np.random.default_rng(7)
    x = rng.uniform(0, 1, (1, 33, 47, 3)).astype(np.float32)
    ctx = binding.Context(0)
    ls, g = _run(ctx, x, x.copy(), 0.2)
    assert ls[0] == 0.0 and ls[1] / x.size == pytest.approx(1.0, abs=1e-6)
    assert np.abs(g).max() <= 1e-6 / x.size * 50           # SSIM is stationary at x == y; sign(0) = 0
    # lambda = 0: the gradient of splx_l1_loss_grad, bit for bit
    y = rng.uniform(0, 1, x.shape).astype(np.float32)
    ls0, g0 = _run(ctx, x, y, 0.0)
    xd, yd = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
    g1 = torch.empty_like(xd); l1 = torch.zeros(1, dtype=torch.float64, device="cuda")
    ctx.l1_loss_grad(xd, yd, g1, l1)
    assert np.array_equal(g0.astype(np.float32), g1.cpu().numpy())
    assert ls0[0] == pytest.approx(float(l1.item()), rel=1e-6)


def test_training_iteration_with_the_dssim_term_against_the_oracle():
    """splx_iteration with lambda_dssim = 0.2 (compose -> L_RGB + lambda L_D-SSIM -> compose backward -> raster and
    projection backward) on the configs[1] recipe shrunk: image, both loss terms and every parameter gradient."""
    sc = scenes.small_aerial()
    cam = sc.cameras[0]
    tr = G.make_trainer(sc)
    tr.lambda_dssim = od.LAMBDA
    plan = tr.make_plan([cam])
    target = torch.from_numpy(sc.targets[0]).cuda()[None]
    img = tr.iteration_fused(plan, target).clone()
    torch.cuda.synchronize()
    res = oracle.forward(sc.partitions(), cam.as_array(), sc.sh_degree, sc.bg)
    frag = np.zeros(res.image.shape[:2], bool)
    for pa in res.partials:
        frag |= pa.margin < G.FRAGILE_MARGIN
    ok = G.close(G.np32(img[0]).astype(np.float64), res.image).all(-1)
    assert (~(ok | frag)).sum() == 0
    L, l1, m, g_image = od.loss(res.image, sc.targets[0], od.LAMBDA)
    ls = tr.loss_sum.cpu().numpy()
    assert ls[0] / res.image.size == pytest.approx(l1, rel=1e-5)
    assert ls[1] / res.image.size == pytest.approx(m, abs=1e-5)
    g_gpu = G.np32(tr._g_images[0]).astype(np.float64)
    assert G.grad_close(g_gpu[~frag], g_image[~frag]) <= 1e-3
    oracle.backward(sc.partitions(), cam.as_array(), sc.sh_degree, res, g_image, sc.bg)
    for key in scenes.PARAM_KEYS:
        got = G.np32(tr.grads[key]).astype(np.float64)
        ref = np.concatenate([g[key].reshape(-1) for g in res.grads])
        assert G.rel_l2(got, ref) <= 1e-3, (key, G.rel_l2(got, ref))
    # and the term changes the gradient: lambda = 0 gives a different one
    sh_grad = tr.grads["sh"].clone()
    tr.lambda_dssim = 0.0
    tr.iteration_fused(plan, target)
    torch.cuda.synchronize()
    assert float((tr.grads["sh"] - sh_grad).abs().max()) > 1e-3 * float(sh_grad.abs().max())
