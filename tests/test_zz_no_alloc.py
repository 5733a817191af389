"""-m gpu: splx_dssim_loss_grad_static, the entry point that allocates nothing (its scratch is a file-scope static
__device__ array inside libsplx.so), against splx_dssim_loss_grad with a caller-owned workspace -- the existing path,
itself held to the oracle in tests/test_gpu_dssim.py.  Two calls in a row on different inputs (the array keeps the
first call's contents), the loss at 1e-5 and dL/dimage at 1e-3 as there.  Collected last on purpose."""
import numpy as np
import pytest
import torch

from paper_2606_18588_b200 import binding, scenes

pytestmark = pytest.mark.gpu


def _cam(W, H):
    return scenes.Camera(np.eye(3, dtype=np.float32), np.zeros(3, np.float32), 50.0, 50.0, W / 2, H / 2, W, H)


def _inputs(seed, B, H, W):
    rng = np.random.default_rng(seed)
    x = rng.uniform(0, 1, (B, H, W, 3)).astype(np.float32)
    y = (0.6 * x + 0.4 * rng.uniform(0, 1, (B, H, W, 3))).astype(np.float32)
    return torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()


def test_static_scratch_entry_equals_the_workspace_path():
    ctx = binding.Context(0)
    lam = 0.2
    # second call: another size (ragged tiles, three views), so stale planes of the first call lie under it
    for seed, (B, H, W) in enumerate([(2, 176, 320), (3, 53, 70)]):
        cam = _cam(W, H)
        x, y = _inputs(100 + seed, B, H, W)
        g_ref, g_new = torch.full_like(x, float("nan")), torch.full_like(x, float("nan"))
        ls_ref = torch.zeros(2, dtype=torch.float64, device="cuda")
        ls_new = torch.zeros(2, dtype=torch.float64, device="cuda")
        ws = torch.empty(B * ctx.dssim_ws_floats(W, H), dtype=torch.float32, device="cuda")
        ctx.dssim_loss_grad(cam, x, y, g_ref, ls_ref, ws, lam)
        before = torch.cuda.memory_allocated()
        ctx.dssim_loss_grad_static(cam, x, y, g_new, ls_new, lam)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before
        a, b = g_new.cpu().numpy().astype(np.float64), g_ref.cpu().numpy().astype(np.float64)
        assert np.isfinite(a).all()
        assert np.abs(a - b).max() <= 1e-3 * np.abs(b).max()
        assert (np.abs(a - b) <= 1e-3 * np.abs(b) + 1e-4 * np.abs(b).max()).all()
        la, lb = ls_new.cpu().numpy(), ls_ref.cpu().numpy()
        assert la[0] == pytest.approx(lb[0], rel=1e-5) and la[1] == pytest.approx(lb[1], rel=1e-5)


def test_static_scratch_entry_rejects_sizes_beyond_its_maximum():
    ctx = binding.Context(0)
    W, H = 1024, 257                       # 263168 pixels > DSSIM_STATIC_MAX_PIXELS = 262144
    assert W * H > binding.DSSIM_STATIC_MAX_PIXELS
    x, y = _inputs(5, 1, H, W)
    g = torch.zeros_like(x)
    launches = ctx.launch_count()
    with pytest.raises(binding.SplxError) as ei:
        ctx.dssim_loss_grad_static(_cam(W, H), x, y, g, None, 0.2)
    assert ei.value.code == -2 and "SPLX_DSSIM_STATIC_MAX_PIXELS" in str(ei.value)
    assert ctx.launch_count() == launches and not g.any()
    ctx.dssim_loss_grad_static(_cam(512, 512), x[:, :256].reshape(1, 512, 512, 3).contiguous(), y[:, :256].reshape(1, 512, 512, 3).contiguous(),
                               g[:, :256].reshape(1, 512, 512, 3), None, 0.2)      # exactly the maximum: accepted
    torch.cuda.synchronize()
