"""Seeded synthetic scenes, cameras, targets and partitions.

This module holds none of the method's arithmetic (no projection, sorting,
blending, composition, gradients or optimiser): it only draws inputs with the
shapes, sizes and value distributions of BASELINE.json's configs (recipe in
DESIGN.md "Input recipe", after SURVEY.md s8(d)) and orders the Gaussians so
that each partition (one "simulated rank") is a contiguous
slice.  It serves both the CUDA path and the oracle; it imports neither.

MatrixCity and trained Gaussians are not available here; these
scenes stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SH0 = 0.28209479177387814  # value of the constant basis function; used only to
                           # turn a target colour into a degree-0 coefficient
PARAM_KEYS = ("mean", "log_scale", "quat", "opacity_logit", "sh")
PARAM_WIDTH = {"mean": 3, "log_scale": 3, "quat": 4, "opacity_logit": 1, "sh": 48}


@dataclass
class Camera:
    R: np.ndarray          # [3,3] row-major, p_cam = R @ mean + t
    t: np.ndarray          # [3]
    fx: float
    fy: float
    cx: float
    cy: float
    width: int
    height: int
    near_z: float = 0.2

    def as_array(self) -> np.ndarray:
        """The 19-double packing both sides unpack: R, t, fx, fy, cx, cy, W, H, near."""
        a = np.zeros(19, dtype=np.float64)
        a[0:9] = np.asarray(self.R, np.float32).astype(np.float64).reshape(9)
        a[9:12] = np.asarray(self.t, np.float32).astype(np.float64).reshape(3)
        a[12:16] = np.asarray([self.fx, self.fy, self.cx, self.cy], np.float32).astype(np.float64)
        a[16:19] = (self.width, self.height, np.float64(np.float32(self.near_z)))
        return a


@dataclass
class Scene:
    name: str
    params: dict            # PARAM_KEYS -> float32 arrays, ordered by partition
    part_offsets: np.ndarray  # int64 [K+1]
    cameras: list           # B cameras
    targets: list           # B float32 [H,W,3]
    sh_degree: int
    bg: tuple = (0.0, 0.0, 0.0)
    meta: dict = field(default_factory=dict)

    @property
    def K(self) -> int:
        return len(self.part_offsets) - 1

    @property
    def N(self) -> int:
        return int(self.part_offsets[-1])

    def partition(self, k: int) -> dict:
        a, b = int(self.part_offsets[k]), int(self.part_offsets[k + 1])
        return {key: self.params[key][a:b] for key in PARAM_KEYS}

    def partitions(self) -> list:
        return [self.partition(k) for k in range(self.K)]


def look_at(position, target, up=(0.0, 0.0, 1.0)):
    """World->camera rotation (rows right, down, forward) and translation."""
    position = np.asarray(position, np.float64)
    fwd = np.asarray(target, np.float64) - position
    fwd /= np.linalg.norm(fwd)
    right = np.cross(fwd, np.asarray(up, np.float64))
    if np.linalg.norm(right) < 1e-9:
        right = np.array([1.0, 0.0, 0.0])
    right /= np.linalg.norm(right)
    down = np.cross(fwd, right)
    R = np.stack([right, down, fwd])
    t = -R @ position
    return R.astype(np.float32), t.astype(np.float32)


def aerial_camera(width, height, fov_deg, altitude, pitch_deg, yaw_deg, target=(0.0, 0.0, 0.0)):
    """Camera at `altitude` above `target`, looking down at `pitch` below horizontal."""
    th, ps = np.deg2rad(pitch_deg), np.deg2rad(yaw_deg)
    dist = altitude / np.sin(th)
    pos = np.asarray(target, np.float64) + dist * np.array(
        [-np.cos(th) * np.cos(ps), -np.cos(th) * np.sin(ps), np.sin(th)])
    R, t = look_at(pos, target)
    f = 0.5 * width / np.tan(0.5 * np.deg2rad(fov_deg))
    return Camera(R, t, f, f, width / 2.0, height / 2.0, width, height)


def street_camera(width, height, fov_deg, position, yaw_deg, pitch_deg=0.0):
    """Street-level camera (the street scenes, where walls saturate whole partitions): at `position`,
    looking along `yaw` at `pitch` above the horizon."""
    ps, th = np.deg2rad(yaw_deg), np.deg2rad(pitch_deg)
    pos = np.asarray(position, np.float64)
    tgt = pos + np.array([np.cos(th) * np.cos(ps), np.cos(th) * np.sin(ps), np.sin(th)])
    R, t = look_at(pos, tgt)
    f = 0.5 * width / np.tan(0.5 * np.deg2rad(fov_deg))
    return Camera(R, t, f, f, width / 2.0, height / 2.0, width, height)


def _rand_quat(rng, n):
    q = rng.standard_normal((n, 4)).astype(np.float32)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    return q


def _order_by_partition(params, part_id, K):
    order = np.argsort(part_id, kind="stable")
    counts = np.bincount(part_id, minlength=K)
    offs = np.zeros(K + 1, np.int64)
    offs[1:] = np.cumsum(counts)
    return {k: np.ascontiguousarray(v[order]) for k, v in params.items()}, offs


def grid_partition(mean, lo, hi, gx, gy):
    """Half-open xy grid cells; outermost cells extend to +-inf (reading s22)."""
    ix = np.clip(np.floor((mean[:, 0] - lo[0]) / (hi[0] - lo[0]) * gx).astype(np.int64), 0, gx - 1)
    iy = np.clip(np.floor((mean[:, 1] - lo[1]) / (hi[1] - lo[1]) * gy).astype(np.int64), 0, gy - 1)
    return iy * gx + ix


def kd_partition(mean, K):
    """"recursive binary splitting akin to a KD-tree, selecting the axis with the largest extent and
    splitting at the median Gaussian position at each level so that the Gaussian counts across partitions remain
    balanced".  K must be a power of two.  Returns part_id[n] in [0, K); leaves are numbered left to right, the lower
    half of a split (ties by index, so the counts of the two halves differ by at most one) first."""
    assert K >= 1 and (K & (K - 1)) == 0, "KD partitions come in powers of two"
    mean = np.asarray(mean)
    part_id = np.zeros(mean.shape[0], np.int64)
    cells = [np.arange(mean.shape[0])]
    while len(cells) < K:
        nxt = []
        for idx in cells:
            if idx.size == 0:
                nxt += [idx, idx]
                continue
            pts = mean[idx]
            axis = int(np.argmax(pts.max(0) - pts.min(0)))
            order = np.argsort(pts[:, axis], kind="stable")
            half = (idx.size + 1) // 2
            nxt += [idx[order[:half]], idx[order[half:]]]
        cells = nxt
    for k, idx in enumerate(cells):
        part_id[idx] = k
    return part_id


def imbalance_ratio(part_offsets):
    """N_max / N_mean - 1 over the partitions."""
    counts = np.diff(np.asarray(part_offsets, np.float64))
    return float(counts.max() / counts.mean() - 1.0)


def partition_aabbs(params, part_offsets, inflate_sigma=3.0):
    """Axis-aligned box of every partition (partitions are AABBs): the bounding box of
    its Gaussians' supports, a Gaussian's support being its mean +- inflate_sigma x its largest scale (reading
    s21; inflate_sigma = 0 gives the box of the means).  Static input of the geometric visibility
    prediction; an empty partition gets the degenerate box lo = hi = 0 (callers drop it from the participants)."""
    K = len(part_offsets) - 1
    lo = np.zeros((K, 3), np.float32)
    hi = np.zeros((K, 3), np.float32)
    on_device = not isinstance(params["mean"], np.ndarray)      # torch tensors of a device-generated scene
    for k in range(K):
        a, b = int(part_offsets[k]), int(part_offsets[k + 1])
        if b > a and on_device:
            m = params["mean"].reshape(-1, 3)[a:b].double()
            r = inflate_sigma * params["log_scale"].reshape(-1, 3)[a:b].double().max(1).values.exp()[:, None]
            lo[k] = np.floor((m - r).min(0).values.cpu().numpy() * 1024) / 1024
            hi[k] = np.ceil((m + r).max(0).values.cpu().numpy() * 1024) / 1024
        elif b > a:
            m = params["mean"][a:b].astype(np.float64)
            r = inflate_sigma * np.exp(params["log_scale"][a:b].astype(np.float64).max(1))[:, None]
            lo[k] = np.floor((m - r).min(0) * 1024) / 1024        # outward rounding to a float32-exact grid
            hi[k] = np.ceil((m + r).max(0) * 1024) / 1024
    return lo, hi


def partition_max_scale(params, part_offsets):
    """Largest scale exp(log_scale) of every partition (0 for an empty one), rounded up to float32."""
    return partition_boxes(params, part_offsets, sub=1)[2]


def partition_boxes(params, part_offsets, sub=1):
    """(lo, hi, max_scale, box_part): a cover of every partition by boxes of MEANS -- the static input of the CONSERVATIVE
    geometric visibility prediction (Trainer.set_aabbs, splx_footprint_margin; reading s21).  sub = 1: one box per
    partition, the bounding box of its Gaussians' means.  sub > 1: that box is cut into sub x sub equal cells in xy and
    every non-empty cell gives the bounding box of the means inside it, so that a far corner of a large partition no
    longer decides the margin of all of it, and one outlier in scale only widens its own cell.  max_scale[j]: the
    largest scale exp(log_scale) among the Gaussians of box j (rounded up to float32); box_part[j]: its partition.
    Boxes are rounded outward to a float32-exact grid.  No arithmetic of the method: input statistics only."""
    K = len(part_offsets) - 1
    los, his, mss, bps = [], [], [], []
    on_device = not isinstance(params["mean"], np.ndarray)
    for k in range(K):
        a, b = int(part_offsets[k]), int(part_offsets[k + 1])
        if b <= a:
            if sub == 1:       # keep one (degenerate) box per partition so that box index == partition index
                los.append(np.zeros(3)); his.append(np.zeros(3)); mss.append(0.0); bps.append(k)
            continue
        if on_device:
            import torch
            m = params["mean"].reshape(-1, 3)[a:b]
            s = params["log_scale"].reshape(-1, 3)[a:b].max(1).values
            lo_k, hi_k = m.min(0).values, m.max(0).values
            if sub == 1:
                cell = torch.zeros(b - a, dtype=torch.int64, device=m.device)
            else:
                ext = torch.clamp(hi_k - lo_k, min=1e-6)
                ix = torch.clamp(((m[:, 0] - lo_k[0]) / ext[0] * sub).long(), 0, sub - 1)
                iy = torch.clamp(((m[:, 1] - lo_k[1]) / ext[1] * sub).long(), 0, sub - 1)
                cell = iy * sub + ix
            nc = sub * sub
            big = torch.finfo(torch.float32).max
            clo = torch.full((nc, 3), big, device=m.device).scatter_reduce(0, cell[:, None].expand(-1, 3), m, "amin")
            chi = torch.full((nc, 3), -big, device=m.device).scatter_reduce(0, cell[:, None].expand(-1, 3), m, "amax")
            cms = torch.full((nc,), -big, device=m.device).scatter_reduce(0, cell, s, "amax")
            cnt = torch.bincount(cell, minlength=nc).cpu().numpy()
            clo, chi, cms = clo.double().cpu().numpy(), chi.double().cpu().numpy(), cms.double().cpu().numpy()
        else:
            m = params["mean"][a:b].astype(np.float64)
            s = params["log_scale"][a:b].astype(np.float64).max(1)
            lo_k, hi_k = m.min(0), m.max(0)
            if sub == 1:
                cell = np.zeros(b - a, np.int64)
            else:
                ext = np.maximum(hi_k - lo_k, 1e-6)
                ix = np.clip(((m[:, 0] - lo_k[0]) / ext[0] * sub).astype(np.int64), 0, sub - 1)
                iy = np.clip(((m[:, 1] - lo_k[1]) / ext[1] * sub).astype(np.int64), 0, sub - 1)
                cell = iy * sub + ix
            nc = sub * sub
            cnt = np.bincount(cell, minlength=nc)
            clo = np.full((nc, 3), np.inf); chi = np.full((nc, 3), -np.inf); cms = np.full(nc, -np.inf)
            np.minimum.at(clo, cell, m); np.maximum.at(chi, cell, m); np.maximum.at(cms, cell, s)
        for c in range(nc):
            if cnt[c] == 0:
                continue
            los.append(np.floor(clo[c] * 1024) / 1024)        # outward rounding to a float32-exact grid
            his.append(np.ceil(chi[c] * 1024) / 1024)
            mss.append(float(np.nextafter(np.float32(np.exp(np.float64(cms[c]))), np.float32(np.inf))))
            bps.append(k)
    return (np.asarray(los, np.float32).reshape(-1, 3), np.asarray(his, np.float32).reshape(-1, 3),
            np.asarray(mss, np.float32), np.asarray(bps, np.int32))


def tiny(seed=0, n=4096, size=128, f=150.0, K=2, sh_degree=0):
    """BASELINE.json configs[0]: world frame = camera frame, K contiguous depth chunks."""
    rng = np.random.default_rng(seed)
    mean = np.empty((n, 3), np.float32)
    mean[:, 0:2] = rng.uniform(-1, 1, (n, 2))
    mean[:, 2] = rng.uniform(2, 6, n)
    params = dict(
        mean=mean,
        log_scale=rng.normal(-3.0, 0.3, (n, 3)).astype(np.float32),
        quat=_rand_quat(rng, n),
        opacity_logit=rng.normal(0.0, 1.0, n).astype(np.float32),
        sh=np.zeros((n, 16, 3), np.float32),
    )
    colour = rng.uniform(0, 1, (n, 3))
    params["sh"][:, 0, :] = ((colour - 0.5) / SH0).astype(np.float32)
    if sh_degree > 0:
        nsh = (sh_degree + 1) ** 2
        params["sh"][:, 1:nsh, :] = rng.normal(0, 0.2, (n, nsh - 1, 3)).astype(np.float32)
    # K contiguous chunks of the depth-sorted list (depth = camera z = mean z here)
    rank = np.argsort(np.argsort(mean[:, 2], kind="stable"), kind="stable")
    part_id = np.minimum(rank * K // n, K - 1)
    order = np.argsort(mean[:, 2], kind="stable")
    params = {k: np.ascontiguousarray(v[order]) for k, v in params.items()}
    part_id = part_id[order]
    offs = np.zeros(K + 1, np.int64)
    offs[1:] = np.cumsum(np.bincount(part_id, minlength=K))
    cam = Camera(np.eye(3, dtype=np.float32), np.zeros(3, np.float32), f, f, size / 2.0, size / 2.0,
                 size, size)
    target = np.random.default_rng(seed + 1).uniform(0, 1, (size, size, 3)).astype(np.float32)
    return Scene("tiny", params, offs, [cam], [target], sh_degree,
                 meta=dict(seed=seed, config="configs[0]"))


def aerial(seed=0, n=1_000_000, width=1920, height=1080, extent=(100.0, 100.0, 20.0), grid=(2, 2),
           altitude=80.0, pitch_deg=45.0, fov_deg=60.0, log_scale_mu=-2.5, log_scale_sigma=0.5,
           sh_degree=3, n_views=1, name="aerial_1M", partition="grid"):
    """BASELINE.json configs[1]: uniform box, K = grid xy partitions, aerial camera."""
    rng = np.random.default_rng(seed)
    ex, ey, ez = extent
    mean = np.empty((n, 3), np.float32)
    mean[:, 0] = rng.uniform(-ex / 2, ex / 2, n)
    mean[:, 1] = rng.uniform(-ey / 2, ey / 2, n)
    mean[:, 2] = rng.uniform(0, ez, n)
    params = dict(
        mean=mean,
        log_scale=rng.normal(log_scale_mu, log_scale_sigma, (n, 3)).astype(np.float32),
        quat=_rand_quat(rng, n),
        opacity_logit=rng.normal(0.0, 1.0, n).astype(np.float32),
        sh=rng.normal(0.0, 0.2, (n, 16, 3)).astype(np.float32),
    )
    K = grid[0] * grid[1]
    if partition == "kd":        # the paper's own partitioner (L480) instead of BASELINE.json's uniform grid
        part_id = kd_partition(mean, K)
    else:
        part_id = grid_partition(mean, (-ex / 2, -ey / 2), (ex / 2, ey / 2), grid[0], grid[1])
    params, offs = _order_by_partition(params, part_id, K)
    crng = np.random.default_rng(seed + 2)
    cams, targets = [], []
    for b in range(n_views):
        yaw = crng.uniform(0, 360)
        cams.append(aerial_camera(width, height, fov_deg, altitude, pitch_deg, yaw))
        targets.append(np.random.default_rng(seed + 1 + 1000 * b)
                       .uniform(0, 1, (height, width, 3)).astype(np.float32))
    return Scene(name, params, offs, cams, targets, sh_degree,
                 meta=dict(seed=seed, config="configs[1]", grid=grid, extent=extent))


def city(seed=0, n=10_000_000, width=1920, height=1080, extent=500.0, n_buildings=200, grid=(4, 2),
         altitude=120.0, pitch_deg=45.0, fov_deg=60.0, height_range=(5.0, 50.0), sh_degree=3,
         n_views=4, name="city_10M", street=False):
    """BASELINE.json configs[2]: 70 % of the means on building surfaces (roof + 4 walls,
    area-weighted, N(0, 0.1 m) jitter), 30 % on the ground plane; K = grid partitions."""
    rng = np.random.default_rng(seed)
    half = extent / 2
    nb = n_buildings
    bc = rng.uniform(-half, half, (nb, 2))
    bs = rng.uniform(10.0, 40.0, (nb, 2))
    bh = rng.uniform(height_range[0], height_range[1], nb)
    n_b = int(0.7 * n)
    n_g = n - n_b
    # faces per building: roof, +x wall, -x wall, +y wall, -y wall
    area = np.stack([bs[:, 0] * bs[:, 1], bs[:, 1] * bh, bs[:, 1] * bh, bs[:, 0] * bh, bs[:, 0] * bh], 1)
    prob = (area / area.sum()).reshape(-1)
    face = rng.choice(nb * 5, size=n_b, p=prob)
    b, f = face // 5, face % 5
    a = rng.uniform(-0.5, 0.5, n_b)
    c = rng.uniform(0.0, 1.0, n_b)
    x = np.where(f == 0, a * bs[b, 0], np.where(f == 1, 0.5 * bs[b, 0], np.where(f == 2, -0.5 * bs[b, 0], a * bs[b, 0])))
    y = np.where(f == 0, (c - 0.5) * bs[b, 1], np.where(f <= 2, a * bs[b, 1], np.where(f == 3, 0.5 * bs[b, 1], -0.5 * bs[b, 1])))
    z = np.where(f == 0, bh[b], c * bh[b])
    mean = np.empty((n, 3), np.float32)
    mean[:n_b, 0] = bc[b, 0] + x
    mean[:n_b, 1] = bc[b, 1] + y
    mean[:n_b, 2] = z
    mean[:n_b] += rng.normal(0, 0.1, (n_b, 3)).astype(np.float32)
    mean[n_b:, 0:2] = rng.uniform(-half, half, (n_g, 2))
    mean[n_b:, 2] = rng.normal(0, 0.05, n_g)
    sp_b = 1.0 / np.sqrt(n_b / area.sum())
    sp_g = 1.0 / np.sqrt(n_g / (extent * extent))
    log_scale = np.empty((n, 3), np.float32)
    log_scale[:n_b] = rng.normal(np.log(1.5 * sp_b), 0.5, (n_b, 3))
    log_scale[n_b:] = rng.normal(np.log(1.0 * sp_g), 0.5, (n_g, 3))
    logit = np.empty(n, np.float32)
    logit[:n_b] = rng.normal(2.0, 1.0, n_b)
    logit[n_b:] = rng.normal(0.0, 1.0, n_g)
    params = dict(mean=mean, log_scale=log_scale, quat=_rand_quat(rng, n), opacity_logit=logit,
                  sh=rng.normal(0.0, 0.2, (n, 16, 3)).astype(np.float32))
    K = grid[0] * grid[1]
    part_id = grid_partition(mean, (-half, -half), (half, half), grid[0], grid[1])
    params, offs = _order_by_partition(params, part_id, K)
    crng = np.random.default_rng(seed + 2)
    cams, targets = [], []
    for v in range(n_views):
        tgt = np.append(crng.uniform(-0.4 * extent, 0.4 * extent, 2), 0.0)
        yaw = crng.uniform(0, 360)
        if street:   # the same seeded spots, seen from 1.7 m above the ground looking along the yaw (street scenes, L296)
            while np.any((np.abs(tgt[:2] - bc) < 0.5 * bs + 2.0).all(1)):      # not inside (or 2 m from) a building
                tgt = np.append(crng.uniform(-0.4 * extent, 0.4 * extent, 2), 0.0)
            cams.append(street_camera(width, height, fov_deg, (tgt[0], tgt[1], 1.7), yaw, 5.0))
        else:
            cams.append(aerial_camera(width, height, fov_deg, altitude, pitch_deg, yaw, tgt))
        targets.append(np.random.default_rng(seed + 1 + 1000 * v)
                       .uniform(0, 1, (height, width, 3)).astype(np.float32))
    return Scene(name, params, offs, cams, targets, sh_degree,
                 meta=dict(seed=seed, config="configs[2]", grid=grid, extent=extent, street=street))


def small_aerial(seed=0, n=20_000, width=320, height=176, K=(2, 2), sh_degree=3):
    """configs[1] shrunk for CPU tests and element-by-element parity: same recipe,
    fewer Gaussians, a smaller image (not a multiple of 16 high -> ragged tile row)
    and scales enlarged so the per-pixel list lengths stay comparable."""
    return aerial(seed=seed, n=n, width=width, height=height, grid=K, sh_degree=sh_degree,
                  log_scale_mu=-0.9, fov_deg=60.0, name=f"aerial_{n}")


def small_city(seed=0, n=30_000, width=320, height=176, n_views=4, grid=(4, 2)):
    """configs[2] shrunk for CPU tests and element-by-element parity: same recipe on a 120 m block with 12
    buildings, B views looking at different parts of it (so that a view touches only some partitions)."""
    return city(seed=seed, n=n, width=width, height=height, extent=120.0, n_buildings=12, grid=grid,
                altitude=35.0, height_range=(5.0, 25.0), n_views=n_views, name=f"city_{n}")


def small_blocks(seed=0, n=24_000, width=320, height=176, n_views=6, grid=(4, 2), extent=(240.0, 120.0, 6.0),
                 altitude=22.0, pitch_deg=62.0):
    """A wide, flat configs[1]-style box cut into grid cells, seen by B low cameras that each look at a
    different spot: a view touches only one to three partitions, so conflict-free buckets
    with several views exist.  Scales are set from the point spacing so that lists stay short."""
    sc = aerial(seed=seed, n=n, width=width, height=height, extent=extent, grid=grid, sh_degree=3, n_views=0,
                log_scale_mu=float(np.log(0.9 * np.sqrt(extent[0] * extent[1] / n))), log_scale_sigma=0.25,
                name=f"blocks_{n}")
    crng = np.random.default_rng(seed + 2)
    for v in range(n_views):
        tgt = (crng.uniform(-0.42, 0.42) * extent[0], crng.uniform(-0.35, 0.35) * extent[1], 0.0)
        sc.cameras.append(aerial_camera(width, height, 60.0, altitude, pitch_deg, crng.uniform(0, 360), tgt))
        sc.targets.append(np.random.default_rng(seed + 1 + 1000 * v).uniform(0, 1, (height, width, 3)).astype(np.float32))
    return sc


def city_device(seed=0, n=40_000_000, width=3840, height=2160, extent=1000.0, n_buildings=800, grid=(4, 4),
                altitude=200.0, pitch_deg=45.0, fov_deg=60.0, height_range=(5.0, 60.0), sh_degree=3, n_views=4,
                name="city_40M", device="cuda"):
    """The configs[2] recipe drawn ON THE DEVICE with a seeded torch generator, for BASELINE.json configs[3]
    (40M Gaussians, 1000 m, 4K views, K = 16) and configs[4] (100M, 2000 m, K = 32): the host arrays would be
    9-24 GB.  Same distributions as `city`; the random streams differ from numpy's, so `city_device(n=10M)` is
    a different (equally distributed) scene than `city()`.  params are CUDA tensors ordered by partition;
    slices are copied back to the host where a test needs them."""
    import torch
    g = torch.Generator(device=device); g.manual_seed(seed)
    f32 = dict(dtype=torch.float32, device=device)
    U = lambda *shape: torch.rand(*shape, generator=g, **f32)
    Nrm = lambda *shape: torch.randn(*shape, generator=g, **f32)
    half = extent / 2
    nb = n_buildings
    bc = (U(nb, 2) * 2 - 1) * half
    bs = 10.0 + 30.0 * U(nb, 2)
    bh = height_range[0] + (height_range[1] - height_range[0]) * U(nb)
    n_b = int(0.7 * n); n_g = n - n_b
    area = torch.stack([bs[:, 0] * bs[:, 1], bs[:, 1] * bh, bs[:, 1] * bh, bs[:, 0] * bh, bs[:, 0] * bh], 1)
    prob = (area / area.sum()).reshape(-1)
    face = torch.multinomial(prob, n_b, replacement=True, generator=g)
    b, f = face // 5, face % 5
    a = U(n_b) - 0.5
    c = U(n_b)
    bsx, bsy, bhh = bs[b, 0], bs[b, 1], bh[b]
    x = torch.where(f == 0, a * bsx, torch.where(f == 1, 0.5 * bsx, torch.where(f == 2, -0.5 * bsx, a * bsx)))
    y = torch.where(f == 0, (c - 0.5) * bsy, torch.where(f <= 2, a * bsy, torch.where(f == 3, 0.5 * bsy, -0.5 * bsy)))
    z = torch.where(f == 0, bhh, c * bhh)
    mean = torch.empty((n, 3), **f32)
    mean[:n_b, 0] = bc[b, 0] + x; mean[:n_b, 1] = bc[b, 1] + y; mean[:n_b, 2] = z
    mean[:n_b] += 0.1 * Nrm(n_b, 3)
    mean[n_b:, 0:2] = (U(n_g, 2) * 2 - 1) * half
    mean[n_b:, 2] = 0.05 * Nrm(n_g)
    del b, f, a, c, x, y, z, bsx, bsy, bhh, face
    sp_b = float(1.0 / np.sqrt(n_b / float(area.sum())))
    sp_g = float(1.0 / np.sqrt(n_g / (extent * extent)))
    log_scale = torch.empty((n, 3), **f32)
    log_scale[:n_b] = np.log(1.5 * sp_b) + 0.5 * Nrm(n_b, 3)
    log_scale[n_b:] = np.log(1.0 * sp_g) + 0.5 * Nrm(n_g, 3)
    logit = torch.empty(n, **f32)
    logit[:n_b] = 2.0 + Nrm(n_b); logit[n_b:] = Nrm(n_g)
    quat = Nrm(n, 4); quat /= quat.norm(dim=1, keepdim=True)
    K = grid[0] * grid[1]
    ix = torch.clamp(torch.floor((mean[:, 0] + half) / extent * grid[0]).long(), 0, grid[0] - 1)
    iy = torch.clamp(torch.floor((mean[:, 1] + half) / extent * grid[1]).long(), 0, grid[1] - 1)
    part_id = iy * grid[0] + ix
    order = torch.argsort(part_id, stable=True)
    counts = torch.bincount(part_id, minlength=K).cpu().numpy()
    offs = np.zeros(K + 1, np.int64); offs[1:] = np.cumsum(counts)
    del ix, iy, part_id
    params = dict(mean=mean[order].contiguous(), log_scale=log_scale[order].contiguous(), quat=quat[order].contiguous(),
                  opacity_logit=logit[order].contiguous())
    del mean, log_scale, quat, logit, order
    params["sh"] = 0.2 * Nrm(n, 16, 3)          # i.i.d.: needs no reordering
    crng = np.random.default_rng(seed + 2)
    cams, targets = [], []
    for v in range(n_views):
        tgt = np.append(crng.uniform(-0.4 * extent, 0.4 * extent, 2), 0.0)
        cams.append(aerial_camera(width, height, fov_deg, altitude, pitch_deg, crng.uniform(0, 360), tgt))
        targets.append(np.random.default_rng(seed + 1 + 1000 * v).uniform(0, 1, (height, width, 3)).astype(np.float32))
    return Scene(name, params, offs, cams, targets, sh_degree,
                 meta=dict(seed=seed, config="configs[3]/[4] recipe, device generator", grid=grid, extent=extent))
