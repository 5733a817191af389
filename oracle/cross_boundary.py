"""Oracle for cross-boundary per-ray filtering -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  PARITY UNPINNED.

PAPER.md L474-L476 (appendix 8.1, Fig. 25): "For two adjacent partitions k and s, let Q_cross denote the set of
Gaussians whose spatial support spans both partitions.  We remove a Gaussian G_i in Q_cross from the ray r of
pixel p if and only if its depth d_i falls within the overlapped depth interval D_overlap and p lies in the
overlapped pixel region Omega_v^k ^ Omega_v^s between the visibility maps of partitions k and s."

The paper defines neither "spatial support" nor D_overlap.  The readings taken are written out
here in fp64 numpy, shared with nothing on the CUDA path:

* support of G_i = the axis-aligned bounding box of its ``sigma``-sigma ellipsoid (sigma = 3, the extent the
  rasteriser uses for the 2-D footprint): half extent along world axis a = sigma * sqrt(Sigma_aa),
  Sigma = R S^2 R^T (L76).  G_i of partition k is in Q_cross(k, s) iff that box meets the box of partition s.
* D^k = the camera-space depth interval of partition k's box under the view k renders (depth is linear, so the
  extremes are at corners); D_overlap(k, s) = D^k ^ D^s, closed.  d_i = the camera-space depth of the mean (L80).
* Omega_v^m = the tile-granular geometric visibility map of ``oracle.visibility.visible_regions`` (DESIGN.md
  s26); "the ray of pixel p" therefore means every pixel of p's tile.  No map given = every tile visible.
* Both partitions must render the same view.  Removal = the Gaussian is left out of that tile's list, forward
  and backward; the order of the others is unchanged.

What IS pinned (tests/test_oracle_cross.py): the ellipsoid extent against sampled ellipsoid points, the depth
interval against sampled box points, and the whole chain against the worked example of Fig. 25 (G3 removed on
r2, kept on r1, global sequence G1-G2-G4 = the single-partition render of those three).  The readings
themselves cannot be pinned to the paper: "parity unpinned".
"""
from __future__ import annotations

import numpy as np

TILE_INVISIBLE = 1


def rotation(quat):
    """Rotation matrices [n,3,3] of un-normalised quaternions (w,x,y,z) (L76; same convention as oracle.project)."""
    q = np.asarray(quat, np.float64)
    q = q / np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((q.shape[0], 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - w * z); R[:, 0, 2] = 2 * (x * z + w * y)
    R[:, 1, 0] = 2 * (x * y + w * z); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - w * x)
    R[:, 2, 0] = 2 * (x * z - w * y); R[:, 2, 1] = 2 * (y * z + w * x); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def covariance(log_scale, quat):
    """Sigma = R S S^T R^T (L76), [n,3,3]."""
    R = rotation(quat)
    S2 = np.exp(2.0 * np.asarray(log_scale, np.float64))
    return np.einsum("nij,nj,nkj->nik", R, S2, R)


def support_half_extent(log_scale, quat, sigma=3.0):
    """Half extents [n,3] of the axis-aligned box around {x: (x-mu)^T Sigma^-1 (x-mu) <= sigma^2}."""
    Sg = covariance(log_scale, quat)
    return sigma * np.sqrt(np.stack([Sg[:, 0, 0], Sg[:, 1, 1], Sg[:, 2, 2]], axis=1))


def cross_sets(mean, log_scale, quat, k, aabb_lo, aabb_hi, sigma=3.0):
    """Gaussians of partition k against all K boxes.  Returns (member[n,K] bool, margin[n,K]): member[i,s] iff
    s != k and the support box of G_i meets box s (closed); margin = the signed overlap that decides it
    (min over axes of the overlap length; >= 0 iff the boxes meet), for the fragile-case protocol of the tests."""
    mean = np.asarray(mean, np.float64)
    lo, hi = np.asarray(aabb_lo, np.float64), np.asarray(aabb_hi, np.float64)
    h = support_half_extent(log_scale, quat, sigma)
    a0, a1 = mean - h, mean + h                                             # [n,3]
    over = np.minimum(a1[:, None, :], hi[None]) - np.maximum(a0[:, None, :], lo[None])   # [n,K,3]
    margin = over.min(axis=2)
    member = margin >= 0
    member[:, k] = False
    return member, margin


def depth_ranges(aabb_lo, aabb_hi, cams, view_of_part):
    """D^k [K,2] = (min, max) camera-space z over the 8 corners of box k under camera view_of_part[k];
    (+inf, -inf) for a partition that renders no view."""
    lo, hi = np.asarray(aabb_lo, np.float64), np.asarray(aabb_hi, np.float64)
    K = lo.shape[0]
    out = np.empty((K, 2))
    for k in range(K):
        v = int(view_of_part[k])
        if v < 0:
            out[k] = (np.inf, -np.inf)
            continue
        cam = np.asarray(cams[v], np.float64).reshape(-1)
        r2, tz = cam[6:9], cam[11]                                          # third row of R, t_z
        zs = [r2 @ np.array([(hi if i & 1 else lo)[k, 0], (hi if i & 2 else lo)[k, 1], (hi if i & 4 else lo)[k, 2]]) + tz
              for i in range(8)]
        out[k] = (min(zs), max(zs))
    return out


def filter_sets(member, depth, k, zr, view_of_part):
    """F[n,K] bool: partitions s for which G_i (of partition k) is removed wherever Omega^s holds:
    G_i in Q_cross(k,s), s renders the view k renders, and d_i in D^k ^ D^s.  The comparison is made on the
    float32 values the kernel compares (a decision, not arithmetic: both sides take it in the same precision)."""
    d = np.asarray(depth, np.float32)
    z = np.asarray(zr, np.float32)
    K = z.shape[0]
    F = np.zeros_like(member, dtype=bool)
    if view_of_part[k] < 0:
        return F
    for s in range(K):
        if s == k or view_of_part[s] != view_of_part[k]:
            continue
        a, b = max(z[k, 0], z[s, 0]), min(z[k, 1], z[s, 1])
        F[:, s] = member[:, s] & (d >= a) & (d <= b)
    return F


def filter_lists(keys, vals, F, tile_state, ntiles):
    """The lists of one partition (``oracle.bin_sort``: keys = tile||depth ascending, vals = local indices) with
    every (Gaussian i, tile t) pair taken out for which some s has F[i,s] and tile t in Omega^s
    (tile_state[s,t] without the INVISIBLE bit; tile_state None = all visible).  Returns keys, vals, ranges."""
    keys, vals = np.asarray(keys, np.uint64), np.asarray(vals, np.int64)
    tile = (keys >> np.uint64(32)).astype(np.int64)
    K = F.shape[1]
    if tile_state is None:
        omega = np.ones((K, ntiles), bool)
    else:
        omega = (np.asarray(tile_state).reshape(K, ntiles) & TILE_INVISIBLE) == 0
    removed = np.zeros(keys.shape[0], bool)
    for j in range(keys.shape[0]):                                          # pair by pair, as the sentence reads
        i, t = vals[j], tile[j]
        removed[j] = bool(np.any(F[i] & omega[:, t]))
    keep = ~removed
    k2, v2, t2 = keys[keep], vals[keep].astype(np.uint32), tile[keep]
    ranges = np.zeros((ntiles, 2), np.uint32)
    for t in np.unique(t2):
        w = np.nonzero(t2 == t)[0]
        ranges[t] = (w[0], w[-1] + 1)
    return k2, v2, ranges
