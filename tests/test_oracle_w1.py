"""Worked example W1 (tests/golden/w1_worked_example.txt): two Gaussians, two partitions,
every value evaluated by hand from PAPER.md Eq.1, Eq.3-5, Eq.6-7.  A wrong sign, a dropped
alpha/T factor or swapped operands anywhere in O1-O8 fails one of these lines."""
import math
import os

import numpy as np
import pytest

import oracle
from tests.common import cam64, gaussians, simple_camera

GOLD = os.path.join(os.path.dirname(__file__), "golden", "w1_worked_example.txt")


def _gold():
    g = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        g[k] = [int(x, 16) if x.startswith("0x") else float(x) for x in v]
    return g


def _parts():
    p0 = gaussians([[0, 0, 4.0]], [0.1], [[1, 0, 0, 0]], [0.0], [[0.9, 0.1, 0.1]])
    p1 = gaussians([[0, 0, 8.0]], [0.2], [[1, 0, 0, 0]], [0.0], [[0.1, 0.9, 0.1]])
    return [p0, p1]


def test_w1_forward_and_backward():
    g = _gold()
    cam = cam64(simple_camera(32, 100.0))
    parts = _parts()
    res = oracle.forward(parts, cam, 0)
    tol = 2e-8
    for k in range(2):
        pr = res.proj[k]
        assert pr.conic_opacity[0, 0] == pytest.approx(g["conic_A"][0], abs=tol)
        assert pr.conic_opacity[0, 2] == pytest.approx(g["conic_A"][0], abs=tol)
        assert pr.conic_opacity[0, 1] == 0
        assert pr.radius[0] == g["radius"][0] and pr.tiles_touched[0] == g["tiles_touched"][0]
        assert list(pr.rect[0]) == [0, 0, 2, 2]
        assert res.bins[k].M == 4
        assert list(res.bins[k].keys >> 32) == [0, 1, 2, 3]
    assert (res.bins[0].keys & 0xFFFFFFFF == g["key_low_bits_g1"][0]).all()
    assert (res.bins[1].keys & 0xFFFFFFFF == g["key_low_bits_g2"][0]).all()
    pa0, pa1 = res.partials
    assert np.allclose(pa0.ct[15, 15, :3], g["C0"], atol=tol) and pa0.ct[15, 15, 3] == pytest.approx(g["T0"][0], abs=tol)
    assert pa0.d[15, 15] == pytest.approx(g["D0"][0], abs=tol)
    assert np.allclose(pa1.ct[15, 15, :3], g["C1"], atol=tol) and pa1.ct[15, 15, 3] == pytest.approx(g["T1"][0], abs=tol)
    assert pa1.d[15, 15] == pytest.approx(g["D1"][0], abs=tol)
    assert np.allclose(res.image[15, 15], g["composite"], atol=tol)
    assert res.T_total[15, 15] == pytest.approx(g["T_total"][0], abs=tol)
    # pixel (8,8): alpha = 9.3e-5 < 1/255 -> skipped
    assert (pa0.ct[8, 8] == [0, 0, 0, 1]).all() and pa0.n_contrib[8, 8] == 0
    # pixel (x=9, y=15): contributes with alpha = 0.01949842
    assert 1 - pa0.ct[15, 9, 3] == pytest.approx(g["alpha_9_15"][0], abs=tol)
    assert pa0.n_contrib[15, 9] == 1
    # symmetry of the footprint about (16,16)
    assert np.allclose(pa0.ct[15, 15], pa0.ct[16, 16]) and np.allclose(pa0.ct[15, 9], pa0.ct[9, 15])

    # backward with dL/dimage = (1,1,1) at pixel (15,15) only
    gi = np.zeros((32, 32, 3)); gi[15, 15] = 1.0
    oracle.backward(parts, cam, 0, res, gi)
    assert np.allclose(res.g_ct[0, 15, 15, :3], 1.0)
    assert res.g_ct[0, 15, 15, 3] == pytest.approx(g["dL_dT0"][0], abs=tol)
    assert np.allclose(res.g_ct[1, 15, 15, :3], g["dL_dC1_scale"][0], atol=tol)
    assert res.g_ct[1, 15, 15, 3] == pytest.approx(g["dL_dT1"][0], abs=tol)
    G = g["G_15_15"][0]
    # dL/dopacity = G dL/dalpha
    assert res.grads2d[0][2][0] == pytest.approx(g["dL_dopacity1"][0], abs=tol)
    assert res.grads2d[0][2][0] / G == pytest.approx(g["dL_dalpha1"][0], abs=tol)
    assert res.grads2d[1][2][0] / G == pytest.approx(g["dL_dalpha2"][0], abs=tol)
    assert res.grads[0]["opacity_logit"][0] == pytest.approx(g["dL_dlogit1"][0], abs=tol)
    # dL/drgb_1 = alpha T = alpha; dL/drgb_2 = T0 * alpha
    a = g["alpha_15_15"][0]
    assert np.allclose(res.grads2d[0][3][0], a, atol=tol)
    assert np.allclose(res.grads2d[1][3][0], g["T0"][0] * a, atol=tol)


def test_w1_slot_swap_gives_same_image():
    cam = cam64(simple_camera(32, 100.0))
    parts = _parts()
    a = oracle.forward(parts, cam, 0)
    b = oracle.forward(parts[::-1], cam, 0)
    assert np.array_equal(a.image, b.image)
    assert (a.order[15, 15] == [0, 1]).all() and (b.order[15, 15] == [1, 0]).all()
