"""Dense fp64 restatement of the path in plain PyTorch CPU ops, for autograd.

Independent of oracle/ (no tiles-as-lists, no hand-derived chain rule, SH built
from associated Legendre functions in spherical angles instead of Cartesian
polynomials).  Every pixel looks at every Gaussian of the partition; the only
inputs it borrows are DECISIONS that are piecewise constant (tile rect
membership, passed in as a boolean mask), so that autograd differentiates
exactly the function PAPER.md Eq.1-5 define.  Used by tests/test_oracle_grad.py
and tests/test_oracle_render.py.  Test infrastructure only.
"""
import math

import torch

TILE = 16


def real_sh_angles(deg, d):
    """Real SH with Condon-Shortley phase, index l*(l+1)+m, from spherical angles.
    d: [...,3] unit vectors.  Returns [..., (deg+1)^2]."""
    x, y, z = d[..., 0], d[..., 1], d[..., 2]
    ct = z.clamp(-1, 1)
    st = torch.sqrt((1 - ct * ct).clamp_min(0))
    phi = torch.atan2(y, x)
    out = []
    for l in range(deg + 1):
        # associated Legendre P_l^m(ct) with CS phase via the standard recurrences
        P = {}
        P[(0, 0)] = torch.ones_like(ct)
        for m in range(1, l + 1):
            P[(m, m)] = -(2 * m - 1) * st * P[(m - 1, m - 1)]
        for m in range(0, l):
            P[(m + 1, m)] = (2 * m + 1) * ct * P[(m, m)]
        for m in range(0, l + 1):
            for ll in range(m + 2, l + 1):
                P[(ll, m)] = ((2 * ll - 1) * ct * P[(ll - 1, m)] - (ll + m - 1) * P[(ll - 2, m)]) / (ll - m)
        for m in range(-l, l + 1):
            am = abs(m)
            N = math.sqrt((2 * l + 1) / (4 * math.pi) * math.factorial(l - am) / math.factorial(l + am))
            if m == 0:
                out.append(N * P[(l, 0)])
            elif m > 0:
                out.append(math.sqrt(2) * N * P[(l, am)] * torch.cos(am * phi))
            else:
                out.append(math.sqrt(2) * N * P[(l, am)] * torch.sin(am * phi))
    return torch.stack(out, -1)


def project_dense(p, cam, sh_degree, dilation=0.3, lim_factor=1.3):
    """p: dict of float64 tensors. cam: dict(R,t,fx,fy,cx,cy,W,H).  Returns 2-D attributes."""
    R, t = cam["R"], cam["t"]
    pc = p["mean"] @ R.T + t
    x, y, z = pc[:, 0], pc[:, 1], pc[:, 2]
    s = torch.exp(p["log_scale"])
    q = p["quat"] / p["quat"].norm(dim=1, keepdim=True)
    w, qx, qy, qz = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    Rot = torch.stack([
        1 - 2 * (qy * qy + qz * qz), 2 * (qx * qy - w * qz), 2 * (qx * qz + w * qy),
        2 * (qx * qy + w * qz), 1 - 2 * (qx * qx + qz * qz), 2 * (qy * qz - w * qx),
        2 * (qx * qz - w * qy), 2 * (qy * qz + w * qx), 1 - 2 * (qx * qx + qy * qy)], -1).reshape(-1, 3, 3)
    Sig = Rot @ torch.diag_embed(s * s) @ Rot.transpose(1, 2)
    limx = lim_factor * cam["W"] / (2 * cam["fx"]); limy = lim_factor * cam["H"] / (2 * cam["fy"])
    tx = torch.clamp(x / z, -limx, limx) * z
    ty = torch.clamp(y / z, -limy, limy) * z
    zero = torch.zeros_like(z)
    J = torch.stack([cam["fx"] / z, zero, -cam["fx"] * tx / (z * z),
                     zero, cam["fy"] / z, -cam["fy"] * ty / (z * z)], -1).reshape(-1, 2, 3)
    Tm = J @ R
    cov = Tm @ Sig @ Tm.transpose(1, 2)
    cov = cov + dilation * torch.eye(2, dtype=cov.dtype)
    conic = torch.linalg.inv(cov)
    u = cam["fx"] * x / z + cam["cx"]; v = cam["fy"] * y / z + cam["cy"]
    o = -(R.T @ t)
    dvec = p["mean"] - o
    dirn = dvec / dvec.norm(dim=1, keepdim=True)
    Y = real_sh_angles(sh_degree, dirn)
    nsh = (sh_degree + 1) ** 2
    rgb = 0.5 + (Y[:, :, None] * p["sh"].reshape(-1, 16, 3)[:, :nsh, :]).sum(1)
    rgb = torch.clamp_min(rgb, 0.0)
    op = torch.sigmoid(p["opacity_logit"])
    return dict(u=u, v=v, z=z, conic=conic, rgb=rgb, op=op)


def render_dense(pr, rect, visible, W, H, alpha_min, alpha_max, T_eps):
    """Every pixel x every Gaussian of the partition (depth order, ties by index).
    rect: int tensor [n,4] tile rect; visible: bool [n].  Returns C[H*W,3], T[H*W], D[H*W]."""
    n = pr["u"].shape[0]
    order = sorted(range(n), key=lambda i: (float(pr["z"][i].detach().float()), i))
    order = torch.tensor(order, dtype=torch.long)
    jj, ii = torch.meshgrid(torch.arange(H), torch.arange(W), indexing="ij")
    px = (ii.reshape(-1) + 0.5).double(); py = (jj.reshape(-1) + 0.5).double()
    tx = (ii.reshape(-1) // TILE); ty = (jj.reshape(-1) // TILE)
    u, v = pr["u"][order], pr["v"][order]
    con = pr["conic"][order]
    dx = u[None, :] - px[:, None]; dy = v[None, :] - py[:, None]
    power = -0.5 * (con[None, :, 0, 0] * dx * dx + con[None, :, 1, 1] * dy * dy) - con[None, :, 0, 1] * dx * dy
    rc = rect[order]
    inrect = ((tx[:, None] >= rc[None, :, 0]) & (tx[:, None] < rc[None, :, 2]) &
              (ty[:, None] >= rc[None, :, 1]) & (ty[:, None] < rc[None, :, 3]) & visible[order][None, :])
    alpha = torch.clamp_max(pr["op"][order][None, :] * torch.exp(power), alpha_max)
    keep = inrect & (power <= 0) & (alpha >= alpha_min)
    alpha = torch.where(keep, alpha, torch.zeros_like(alpha))
    # early exit: sequential scan (decision only; values flow through alpha)
    with torch.no_grad():
        a = alpha.detach()
        Tn = torch.ones(a.shape[0], dtype=a.dtype)
        alive = torch.ones(a.shape[0], dtype=torch.bool)
        live = torch.zeros_like(keep)
        for g in range(n):
            cand = Tn * (1 - a[:, g])
            stop = alive & keep[:, g] & (cand < T_eps)
            alive = alive & ~stop
            take = alive & keep[:, g]
            live[:, g] = take
            Tn = torch.where(take, cand, Tn)
    alpha = torch.where(live, alpha, torch.zeros_like(alpha))
    one_m = 1 - alpha
    Tincl = torch.cumprod(one_m, dim=1)
    Texcl = torch.cat([torch.ones_like(Tincl[:, :1]), Tincl[:, :-1]], 1)
    wgt = alpha * Texcl
    C = wgt @ pr["rgb"][order]
    D = wgt @ pr["z"][order]
    return C, Tincl[:, -1], D


def compose_dense(Cs, Ts, Ds, bg):
    """Eq.5 with the key D/(1-T), stable by partition index; decisions from detached values."""
    K = len(Cs)
    P = Cs[0].shape[0]
    key = torch.stack([torch.where(Ts[k] < 1, Ds[k] / (1 - Ts[k]).clamp_min(1e-300),
                                   torch.full_like(Ts[k], float("inf"))) for k in range(K)], 1).detach()
    perm = torch.argsort(key, dim=1, stable=True)
    Cst = torch.stack(Cs, 1); Tst = torch.stack(Ts, 1)
    Cp = torch.gather(Cst, 1, perm[:, :, None].expand(P, K, 3))
    Tp = torch.gather(Tst, 1, perm)
    Tincl = torch.cumprod(Tp, 1)
    Tfront = torch.cat([torch.ones_like(Tincl[:, :1]), Tincl[:, :-1]], 1)
    img = (Tfront[:, :, None] * Cp).sum(1) + Tincl[:, -1:] * bg[None, :]
    return img, Tincl[:, -1]
