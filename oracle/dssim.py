"""D-SSIM loss term of PAPER.md L95 ("L = L_RGB + lambda L_D-SSIM") -- CPU oracle, TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes driver of ``oracle/dssim_oracle.c`` (plain C, fp64, direct 121-term window loops).  Reading s33 of DESIGN.md:
L_D-SSIM = 1 - mean SSIM, 11 x 11 Gaussian window (sigma 1.5), C1 = 0.01^2, C2 = 0.03^2, zero padding, lambda = 0.2 --
none of which the paper states (parity unpinned against the authors' code; the SSIM definition itself is pinned in
tests/test_oracle_dssim.py).  Never imported by the product package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dssim_oracle.c")
_LIB = os.path.join(_HERE, "libdssim_oracle.so")
_lib = None

LAMBDA = 0.2


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _L():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.orc_ssim.restype = ctypes.c_double
    return _lib


def ssim(image, target, want_map=False, want_grad=True):
    """mean SSIM over H*W*C, optionally the SSIM map and d(mean SSIM)/d(image).  image, target: [H,W,C]."""
    x = np.ascontiguousarray(image, np.float64)
    y = np.ascontiguousarray(target, np.float64)
    assert x.shape == y.shape and x.ndim == 3
    H, W, C = x.shape
    smap = np.zeros_like(x) if want_map else None
    g = np.zeros_like(x) if want_grad else None
    p = lambda a: a.ctypes.data_as(ctypes.c_void_p) if a is not None else None
    m = _L().orc_ssim(W, H, C, p(x), p(y), p(smap), p(g))
    return float(m), smap, g


def loss(image, target, lam=LAMBDA):
    """L = mean|image - target| + lam * (1 - mean SSIM) and dL/d(image).  Returns (L, L1, mean SSIM, grad)."""
    x = np.ascontiguousarray(image, np.float64)
    y = np.ascontiguousarray(target, np.float64)
    diff = x - y
    l1 = float(np.abs(diff).mean())
    g = np.sign(diff) / diff.size
    m, _, gs = ssim(x, y)
    return l1 + lam * (1.0 - m), l1, m, g - lam * gs
