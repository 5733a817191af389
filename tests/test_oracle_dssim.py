"""Pins of the D-SSIM oracle (oracle/dssim_oracle.c; "L = L_RGB + lambda L_D-SSIM", reading s33).
Each pin fails for a plausible mistake: a dropped term of the derivative (central differences, autograd), a wrong
window or padding (scipy's gaussian_filter, the corner closed form), swapped operands (symmetry), a wrong constant
(the constant-image closed form)."""
import numpy as np
import pytest
import torch
from scipy import ndimage

from oracle import dssim

C1, C2 = 0.01 ** 2, 0.03 ** 2


def _images(seed, H=21, W=26, C=3):
    rng = np.random.default_rng(seed)
    return rng.uniform(0, 1, (H, W, C)), rng.uniform(0, 1, (H, W, C))


def test_identical_images_have_ssim_one_and_no_gradient():
    x, _ = _images(0)
    m, smap, g = dssim.ssim(x, x, want_map=True)
    assert m == pytest.approx(1.0, abs=1e-15)
    assert np.allclose(smap, 1.0, atol=1e-14)
    assert np.abs(g).max() < 1e-15              # SSIM is maximal at x == y
    L, l1, ms, gl = dssim.loss(x, x)
    assert L == 0.0 and l1 == 0.0 and np.abs(gl).max() < 1e-15


def test_constant_images_closed_form_interior_and_corner():
    """x = a, y = b everywhere.  Interior (window inside the image): all variances vanish,
    SSIM = (2ab + C1)/(a^2 + b^2 + C1).  Corner pixel: the window mass inside the image is m = (sum_{i>=0} w_i)^2, so
    mu = m a, E[x^2] = m a^2: SSIM = (2 m^2 ab + C1)(2 m(1-m) ab + C2) / ((m^2(a^2+b^2) + C1)(m(1-m)(a^2+b^2) + C2))."""
    a, b = 0.7, 0.4
    H, W = 16, 18
    x = np.full((H, W, 1), a); y = np.full((H, W, 1), b)
    _, smap, _ = dssim.ssim(x, y, want_map=True, want_grad=False)
    assert smap[8, 9, 0] == pytest.approx((2 * a * b + C1) / (a * a + b * b + C1), rel=1e-13)
    w = np.exp(-np.arange(-5, 6) ** 2 / (2 * 1.5 ** 2)); w /= w.sum()
    m = w[5:].sum() ** 2
    s2 = a * a + b * b
    want = (2 * m * m * a * b + C1) * (2 * m * (1 - m) * a * b + C2) / ((m * m * s2 + C1) * (m * (1 - m) * s2 + C2))
    assert smap[0, 0, 0] == pytest.approx(want, rel=1e-12)
    assert smap[H - 1, W - 1, 0] == pytest.approx(want, rel=1e-12)


def test_window_sums_against_scipy_gaussian_filter():
    """The five window sums through a LIBRARY Gaussian filter (sigma 1.5, radius 5 = truncate 3.0, zero padding)."""
    x, y = _images(1)
    f = lambda a: np.stack([ndimage.gaussian_filter(a[..., c], 1.5, mode="constant", cval=0.0, truncate=3.0)
                            for c in range(a.shape[-1])], -1)
    mx, my = f(x), f(y)
    sxx, syy, sxy = f(x * x) - mx * mx, f(y * y) - my * my, f(x * y) - mx * my
    ref = ((2 * mx * my + C1) * (2 * sxy + C2)) / ((mx * mx + my * my + C1) * (sxx + syy + C2))
    m, smap, _ = dssim.ssim(x, y, want_map=True, want_grad=False)
    assert np.allclose(smap, ref, rtol=0, atol=1e-12)
    assert m == pytest.approx(ref.mean(), abs=1e-13)


def test_symmetry_and_bound():
    x, y = _images(2)
    mxy = dssim.ssim(x, y, want_grad=False)[0]
    myx = dssim.ssim(y, x, want_grad=False)[0]
    assert mxy == pytest.approx(myx, abs=1e-14)
    _, smap, _ = dssim.ssim(x, y, want_map=True, want_grad=False)
    assert smap.max() <= 1.0 + 1e-12


def test_gradient_central_differences():
    x, y = _images(3, H=13, W=14, C=2)
    _, _, g = dssim.ssim(x, y)
    h = 1e-6
    rng = np.random.default_rng(4)
    idx = [(0, 0, 0), (12, 13, 1), (0, 13, 0), (6, 7, 1)] + [tuple(rng.integers(0, s) for s in x.shape) for _ in range(40)]
    for i in idx:
        xp, xm = x.copy(), x.copy()
        xp[i] += h; xm[i] -= h
        fd = (dssim.ssim(xp, y, want_grad=False)[0] - dssim.ssim(xm, y, want_grad=False)[0]) / (2 * h)
        assert g[i] == pytest.approx(fd, rel=2e-5, abs=1e-10), i


def test_gradient_against_autograd_of_a_conv2d_restatement():
    """Independent of the hand-derived chain rule: fp64 autograd through torch's conv2d (a library routine)."""
    x, y = _images(5)
    w1 = torch.exp(-torch.arange(-5, 6, dtype=torch.float64) ** 2 / (2 * 1.5 ** 2)); w1 /= w1.sum()
    win = (w1[:, None] * w1[None, :])[None, None].repeat(3, 1, 1, 1)
    X = torch.tensor(x).permute(2, 0, 1)[None].clone().requires_grad_(True)
    Y = torch.tensor(y).permute(2, 0, 1)[None]
    conv = lambda a: torch.nn.functional.conv2d(a, win, padding=5, groups=3)
    mx, my = conv(X), conv(Y)
    sxx, syy, sxy = conv(X * X) - mx * mx, conv(Y * Y) - my * my, conv(X * Y) - mx * my
    S = ((2 * mx * my + C1) * (2 * sxy + C2)) / ((mx * mx + my * my + C1) * (sxx + syy + C2))
    S.mean().backward()
    m, _, g = dssim.ssim(x, y)
    assert m == pytest.approx(float(S.mean().detach()), abs=1e-13)
    assert np.allclose(g, X.grad[0].permute(1, 2, 0).numpy(), rtol=1e-9, atol=1e-15)


def test_loss_combines_l1_and_dssim():
    x, y = _images(6)
    lam = 0.2
    L, l1, m, g = dssim.loss(x, y, lam)
    assert l1 == pytest.approx(np.abs(x - y).mean(), rel=1e-15)
    assert L == pytest.approx(l1 + lam * (1 - m), rel=1e-15)
    _, _, gs = dssim.ssim(x, y)
    assert np.allclose(g, np.sign(x - y) / x.size - lam * gs, atol=1e-18)
    # lambda = 0 is the plain mean-L1 harness loss
    L0, _, _, g0 = dssim.loss(x, y, 0.0)
    assert L0 == l1 and np.array_equal(g0, np.sign(x - y) / x.size)
