"""Pins for oracle O7 (raster backward), O8 (projection backward) and O9 (Adam):
(i) central finite differences of the oracle's own forward, in double;
(ii) float64 autograd on the independent dense restatement (tests/dense_ref.py);
(iii) torch.optim.Adam (library routine) and the first-step closed form.
PAPER.md L184-L190 (gradient through the partial pixel), L95 (all parameters updated)."""
import numpy as np
import pytest
import torch

import oracle
from tests import dense_ref
from tests.common import cam64, random_scene

KEYS = ("mean", "log_scale", "quat", "opacity_logit", "sh")


def _split(p, K):
    n = p["mean"].shape[0]
    cuts = [n * k // K for k in range(K + 1)]
    return [{key: p[key][cuts[k]:cuts[k + 1]] for key in KEYS} for k in range(K)]


def _loss(parts, cam, deg, wimg, wT, bg, cfg):
    res = oracle.forward(parts, cam, deg, bg, cfg)
    return (res.image * wimg).sum() + (res.T_total * wT).sum(), res


@pytest.mark.parametrize("seed,deg,cfg", [(30, 3, oracle.SMOOTH_CFG), (31, 1, oracle.SMOOTH_CFG),
                                          (32, 3, oracle.DEFAULT_CFG)])
def test_full_chain_central_differences(seed, deg, cfg):
    rng = np.random.default_rng(seed)
    n, K, size = 24, 2, 32
    p, cam = random_scene(rng, n, size=size, f=40.0, sh_degree=deg)
    p["sh"][:, 0, 0] -= 2.5  # make some red channels clamp at 0 (masked gradient)
    p["mean"][0] = (np.array([1.9, 0.1, 3.0]) - np.asarray(cam.t, np.float64)) @ np.asarray(cam.R, np.float64)
    # ^ x/z = 0.63 > 1.3 * 16/40 = 0.52: Gaussian 0 sits in the clamped-J region
    camv = cam64(cam)
    parts = _split(p, K)
    wimg = rng.standard_normal((size, size, 3)); wT = rng.standard_normal((size, size))
    bg = (0.2, 0.4, 0.6)
    L0, res = _loss(parts, camv, deg, wimg, wT, bg, cfg)
    oracle.backward(parts, camv, deg, res, wimg, bg, cfg, g_T_total=wT)
    assert any((pr.clamp != 0).any() for pr in res.proj)
    checked = 0
    for k in range(K):
        for key in KEYS:
            g = res.grads[k][key].reshape(-1)
            flat_idx = rng.choice(g.size, min(g.size, 14), replace=False)
            for fi in flat_idx:
                base = parts[k][key]
                h = 1e-6 * max(1.0, abs(base.reshape(-1)[fi]))
                vals = []
                for sgn in (+1, -1):
                    q = [dict(pp) for pp in parts]
                    arr = base.copy(); arr.reshape(-1)[fi] += sgn * h
                    q[k][key] = arr
                    vals.append(_loss(q, camv, deg, wimg, wT, bg, cfg)[0])
                fd = (vals[0] - vals[1]) / (2 * h)
                if cfg is oracle.DEFAULT_CFG:
                    # threshold mode: a decision may flip inside [-h, h]; detect by a second step size
                    vals2 = []
                    for sgn in (+1, -1):
                        q = [dict(pp) for pp in parts]
                        arr = base.copy(); arr.reshape(-1)[fi] += sgn * h / 4
                        q[k][key] = arr
                        vals2.append(_loss(q, camv, deg, wimg, wT, bg, cfg)[0])
                    fd2 = (vals2[0] - vals2[1]) / (h / 2)
                    if abs(fd - fd2) > 1e-4 * max(1e-6, abs(fd)):
                        continue
                assert g[fi] == pytest.approx(fd, rel=2e-5, abs=2e-7), (k, key, fi)
                checked += 1
    assert checked > 80


def _torch_parts(parts):
    return [{k: torch.tensor(np.asarray(v, np.float64), requires_grad=True) for k, v in p.items()}
            for p in parts]


@pytest.mark.parametrize("seed,cfg", [(40, oracle.DEFAULT_CFG), (41, oracle.SMOOTH_CFG)])
def test_gradients_match_fp64_autograd_of_dense_restatement(seed, cfg):
    rng = np.random.default_rng(seed)
    n, K, size, deg = 40, 3, 32, 3
    p, cam = random_scene(rng, n, size=size, f=40.0, sh_degree=deg)
    p["opacity_logit"] += 1.5
    p["sh"][:, 0, 1] -= 2.5
    camv = cam64(cam)
    parts = _split(p, K)
    wimg = rng.standard_normal((size, size, 3)); wT = rng.standard_normal((size, size))
    bg = (0.1, 0.3, 0.5)
    _, res = _loss(parts, camv, deg, wimg, wT, bg, cfg)
    oracle.backward(parts, camv, deg, res, wimg, bg, cfg, g_T_total=wT)

    tparts = _torch_parts(parts)
    cd = dict(R=torch.tensor(np.asarray(cam.R, np.float64)), t=torch.tensor(np.asarray(cam.t, np.float64)),
              fx=cam.fx, fy=cam.fy, cx=cam.cx, cy=cam.cy, W=size, H=size)
    Cs, Ts, Ds = [], [], []
    for k in range(K):
        prd = dense_ref.project_dense(tparts[k], cd, deg)
        C, T, D = dense_ref.render_dense(prd, torch.tensor(res.proj[k].rect), torch.tensor(res.proj[k].radius > 0),
                                         size, size, cfg[0], cfg[1], cfg[2])
        Cs.append(C); Ts.append(T); Ds.append(D)
    img, Tt = dense_ref.compose_dense(Cs, Ts, Ds, torch.tensor(bg, dtype=torch.float64))
    assert np.abs(img.detach().numpy().reshape(size, size, 3) - res.image).max() < 1e-11
    L = (img * torch.tensor(wimg.reshape(-1, 3))).sum() + (Tt * torch.tensor(wT.reshape(-1))).sum()
    L.backward()
    for k in range(K):
        for key in KEYS:
            ref = tparts[k][key].grad.numpy().reshape(res.grads[k][key].shape)
            got = res.grads[k][key]
            if key == "sh":  # only the first (deg+1)^2 coefficients are read
                assert not got[:, (deg + 1) ** 2:].any()
            scale = max(np.abs(ref).max(), 1e-12)
            assert np.abs(got - ref).max() <= 1e-9 * scale, (k, key, np.abs(got - ref).max(), scale)
            assert np.abs(ref).max() > 0


def test_adam_first_step_closed_form_and_torch_optim():
    rng = np.random.default_rng(50)
    n = 257
    p0 = rng.standard_normal(n); g = rng.standard_normal(n) * 10.0 ** rng.uniform(-6, 2, n)
    p = p0.copy(); m = np.zeros(n); v = np.zeros(n)
    oracle.adam(p, g, m, v, lr=1e-2, step=1)
    # first step: m_hat = g, v_hat = g^2 -> delta = -lr g/(|g| + eps)
    assert np.allclose(p - p0, -1e-2 * g / (np.abs(g) + 1e-15), rtol=1e-12, atol=0)
    # 10 steps against the library optimiser, float64
    tp = torch.tensor(p0.copy(), requires_grad=True)
    opt = torch.optim.Adam([tp], lr=3e-3, betas=(0.9, 0.999), eps=1e-15)
    p = p0.copy(); m = np.zeros(n); v = np.zeros(n)
    for step in range(1, 11):
        gs = rng.standard_normal(n) * (1 + 0.1 * step)
        tp.grad = torch.tensor(gs.copy())
        opt.step()
        oracle.adam(p, gs, m, v, lr=3e-3, step=step)
    assert np.allclose(p, tp.detach().numpy(), rtol=1e-12, atol=1e-14)
