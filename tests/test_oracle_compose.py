"""Pins for oracle O4 (global composition, Eq.5) and O6 (its backward,
L186-L188 Eq.6-7): the invariants the paper states (L180: Eq.5 == Eq.2), closed forms,
algebraic properties of 'over', and central finite differences."""
import numpy as np
import pytest

import oracle
from paper_2606_18588_b200 import scenes


def _rand_partials(rng, K, H=8, W=8, frac_empty=0.3):
    ct = np.zeros((K, H, W, 4)); d = np.zeros((K, H, W))
    T = rng.uniform(0.05, 0.95, (K, H, W))
    col = rng.uniform(0, 1, (K, H, W, 3))
    ct[..., :3] = col * (1 - T)[..., None]
    ct[..., 3] = T
    d[:] = rng.uniform(1, 10, (K, H, W)) * (1 - T)
    empty = rng.uniform(size=(K, H, W)) < frac_empty
    ct[empty] = [0, 0, 0, 1]; d[empty] = 0
    return ct, d


def test_k1_is_partial_plus_background():
    # north_star check 1: K=1 composition equals the direct render (+ T bg)
    rng = np.random.default_rng(0)
    ct, d = _rand_partials(rng, 1)
    bg = np.array([0.2, 0.5, 0.7])
    img, Tt, _, _ = oracle.compose(ct, d, bg)
    assert np.allclose(img, ct[0, ..., :3] + ct[0, ..., 3:4] * bg, atol=1e-15)
    assert np.array_equal(Tt, ct[0, ..., 3])


def test_k2_closed_form_and_key_order():
    # C = C_near + T_near C_far, ordered by D/(1-T) whatever the slot
    ct = np.zeros((2, 16, 16, 4)); d = np.zeros((2, 16, 16))
    ct[0, ..., :] = [0.1, 0.2, 0.3, 0.5]; d[0] = 0.5 * 7.0   # mean depth 7
    ct[1, ..., :] = [0.4, 0.0, 0.1, 0.25]; d[1] = 0.75 * 3.0  # mean depth 3 -> in front
    img, Tt, order, _ = oracle.compose(ct, d)
    assert np.allclose(img[0, 0], np.array([0.4, 0.0, 0.1]) + 0.25 * np.array([0.1, 0.2, 0.3]))
    assert Tt[0, 0] == 0.125 and list(order[0, 0]) == [1, 0]
    # un-normalised D would have ordered slot 0 (D=3.5) after slot 1 (D=2.25) too; make a case where
    # only the normalised key (reading s3) is right: faint far partition, solid near one
    ct[0, ..., :] = [0.01, 0.01, 0.01, 0.98]; d[0] = 0.02 * 50.0  # D = 1.0, mean depth 50
    ct[1, ..., :] = [0.5, 0.5, 0.5, 0.1]; d[1] = 0.9 * 5.0         # D = 4.5, mean depth 5
    _, _, order, _ = oracle.compose(ct, d)
    assert list(order[0, 0]) == [1, 0]


def test_contiguous_depth_chunks_reproduce_full_render():
    # north_star check 2 / PAPER.md L180: with partitions = contiguous chunks of the depth-sorted
    # list, composing the K partials reproduces the full-scene render.  Exact (to rounding) with
    # T_eps = 0; with T_eps = 1e-4 bounded by the light the full render drops at its exit.
    for K in (2, 3, 5):
        sc = scenes.tiny(n=3000, size=48, f=56.0, K=K)
        cam = sc.cameras[0].as_array()
        whole = [{k: sc.params[k] for k in scenes.PARAM_KEYS}]
        cfg0 = (1 / 255, 0.99, 0.0, 0.3, 1.3, 0.1)
        full = oracle.forward(whole, cam, 0, cfg=cfg0)
        comp = oracle.forward(sc.partitions(), cam, 0, cfg=cfg0)
        assert np.abs(full.image - comp.image).max() < 1e-13
        assert np.abs(full.T_total - comp.T_total).max() < 1e-13
        # every pixel's order is the chunk order (chunks are depth-separated), empties last
        for k in range(K):
            live = np.stack([pa.ct[..., 3] < 1 for pa in comp.partials], -1)
        o = comp.order
        for r in range(K - 1):
            a, b = o[..., r], o[..., r + 1]
            la = np.take_along_axis(live, a[..., None], -1)[..., 0]
            lb = np.take_along_axis(live, b[..., None], -1)[..., 0]
            assert ((a < b) | ~lb | ~la).all() and (la | ~lb).all()
        full = oracle.forward(whole, cam, 0)
        comp = oracle.forward(sc.partitions(), cam, 0)
        te = full.partials[0].t_exit
        bound = np.where(te >= 0, te, 0.0)[..., None] * full.proj[0].rgb.max() + 1e-13
        assert (np.abs(full.image - comp.image) <= bound).all()
        assert (te >= 0).any()


def test_gradients_of_chunks_sum_to_full_scene_gradient():
    # pin (iii) of SURVEY s8(c): Eq.6-7 + per-partition backward == backward of the full render
    sc = scenes.tiny(n=600, size=32, f=37.0, K=3)
    cam = sc.cameras[0].as_array()
    cfg0 = (1 / 255, 0.99, 0.0, 0.3, 1.3, 0.1)
    whole = [{k: sc.params[k] for k in scenes.PARAM_KEYS}]
    tgt = sc.targets[0]
    full = oracle.iteration(whole, cam, 0, tgt, cfg=cfg0)
    comp = oracle.iteration(sc.partitions(), cam, 0, tgt, cfg=cfg0)
    for key in scenes.PARAM_KEYS:
        cat = np.concatenate([g[key] for g in comp.grads])
        ref = full.grads[0][key]
        assert np.abs(cat - ref).max() <= 1e-9 * max(1e-30, np.abs(ref).max()), key
        assert np.abs(ref).max() > 0


def test_over_is_associative_and_slot_invariant_with_identity():
    rng = np.random.default_rng(1)
    ct, d = _rand_partials(rng, 4)
    bg = np.array([0.3, 0.1, 0.9])
    img, Tt, _, _ = oracle.compose(ct, d, bg)
    perm = [2, 0, 3, 1]
    img2, Tt2, _, _ = oracle.compose(ct[perm], d[perm], bg)
    assert np.allclose(img, img2, atol=1e-15) and np.allclose(Tt, Tt2, atol=1e-15)
    # identity element (C=0, T=1) anywhere changes nothing
    ct5 = np.concatenate([ct[:2], np.broadcast_to([0, 0, 0, 1.0], (1, 8, 8, 4)), ct[2:]])
    d5 = np.concatenate([d[:2], np.zeros((1, 8, 8)), d[2:]])
    img3, Tt3, _, _ = oracle.compose(ct5, d5, bg)
    assert np.allclose(img, img3, atol=1e-15) and np.allclose(Tt, Tt3, atol=1e-15)
    # associativity: merge the two front-most partials of every pixel into one, recompose
    _, _, order, _ = oracle.compose(ct, d, bg)
    H = W = 8
    ii, jj = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    f0, f1 = order[..., 0], order[..., 1]
    A = ct[f0, ii, jj]; B = ct[f1, ii, jj]
    merged = np.concatenate([A[..., :3] + A[..., 3:4] * B[..., :3], A[..., 3:4] * B[..., 3:4]], -1)
    dm = d[f0, ii, jj] + A[..., 3] * d[f1, ii, jj]
    rest = np.stack([ct[order[..., r], ii, jj] for r in (2, 3)])
    drest = np.stack([d[order[..., r], ii, jj] for r in (2, 3)])
    img4, _, _, _ = oracle.compose(np.concatenate([merged[None], rest]), np.concatenate([dm[None], drest]), bg)
    assert np.allclose(img, img4, atol=1e-14)


def test_compose_bwd_closed_forms():
    # loss = sum C with K=2: dL/dT_front = sum C_back (+ T_back sum bg); K=1: dL/dT = <g, bg>
    rng = np.random.default_rng(2)
    ct, d = _rand_partials(rng, 2, frac_empty=0.0)
    d[0] = (1 - ct[0, ..., 3]) * 2.0; d[1] = (1 - ct[1, ..., 3]) * 6.0  # slot 0 in front everywhere
    g = np.ones((8, 8, 3))
    gct = oracle.compose_bwd(ct, d, g)
    assert np.allclose(gct[0, ..., :3], 1.0) and np.allclose(gct[0, ..., 3], ct[1, ..., :3].sum(-1))
    assert np.allclose(gct[1, ..., :3], ct[0, ..., 3:4]) and np.allclose(gct[1, ..., 3], 0.0)
    bg = np.array([0.2, 0.3, 0.4])
    gct = oracle.compose_bwd(ct[:1], d[:1], g, bg)
    assert np.allclose(gct[0, ..., 3], 0.9)
    gct = oracle.compose_bwd(ct, d, g, bg)
    assert np.allclose(gct[1, ..., 3], ct[0, ..., 3] * 0.9)
    assert np.allclose(gct[0, ..., 3], ct[1, ..., :3].sum(-1) + ct[1, ..., 3] * 0.9)


@pytest.mark.parametrize("K", [1, 3, 6])
def test_compose_bwd_central_differences(K):
    rng = np.random.default_rng(3 + K)
    ct, d = _rand_partials(rng, K, H=4, W=4)
    bg = np.array([0.3, 0.6, 0.2])
    gi = rng.standard_normal((4, 4, 3)); gT = rng.standard_normal((4, 4))

    def loss(c):
        img, Tt, _, _ = oracle.compose(c, d, bg)
        return (img * gi).sum() + (Tt * gT).sum()

    gct = oracle.compose_bwd(ct, d, gi, bg, gT)
    h = 1e-6
    idx = [(k, j, i, c) for k in range(K) for j in range(4) for i in range(4) for c in range(4)]
    for k, j, i, c in [idx[t] for t in rng.choice(len(idx), 60, replace=False)]:
        if ct[k, j, i, 3] == 1.0:  # an empty partition sits at key +inf; perturbing T would re-order it
            continue
        p, m = ct.copy(), ct.copy()
        p[k, j, i, c] += h; m[k, j, i, c] -= h
        fd = (loss(p) - loss(m)) / (2 * h)
        assert gct[k, j, i, c] == pytest.approx(fd, rel=1e-6, abs=1e-8)


def test_l1_loss():
    rng = np.random.default_rng(5)
    a = rng.uniform(size=(4, 5, 3)); b = rng.uniform(size=(4, 5, 3)); b[0, 0] = a[0, 0]
    L, g = oracle.l1(a, b)
    assert L == pytest.approx(np.abs(a - b).mean())
    assert np.array_equal(g, np.sign(a - b) / a.size)
