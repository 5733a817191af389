"""Buffer ownership and call sequencing for one training iteration on one B200.

``Trainer`` owns the device memory (parameters, gradients, Adam moments, projected attributes,
binning, partial-pixel buffers) and issues the C-ABI calls of ``include/splx.h`` in the order
of SURVEY.md s3(b).  It performs no arithmetic of the method itself: every step runs in the
CUDA kernels behind ``binding.Context``.  K partitions = K contiguous slices of the SoA.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding
from .scenes import PARAM_KEYS, PARAM_WIDTH

#: conventional 3DGS learning rates (paper silent)
DEFAULT_LR = {"mean": 1.6e-4, "log_scale": 5e-3, "quat": 1e-3, "opacity_logit": 5e-2, "sh": 2.5e-3}


def _flat_layout(n):
    """Offsets (in floats) of the five parameter groups inside one flat buffer, 16-B aligned."""
    offs, cur = {}, 0
    for k in PARAM_KEYS:
        offs[k] = cur
        cur += (n * PARAM_WIDTH[k] + 3) // 4 * 4
    return offs, cur


class Trainer:
    def __init__(self, params: dict, part_offsets, width, height, sh_degree=3, bg=(0.0, 0.0, 0.0),
                 capacity=None, device=0, cfg=None, lr=None):
        self.ctx = binding.Context(device, cfg=cfg)
        dev = self.ctx.device
        self.n = int(params["mean"].shape[0])
        self.K = len(part_offsets) - 1
        self.part_offsets = [int(x) for x in part_offsets]
        self.W, self.H, self.sh_degree, self.bg = int(width), int(height), int(sh_degree), tuple(bg)
        self.lr = dict(DEFAULT_LR if lr is None else lr)
        offs, total = _flat_layout(self.n)
        self._offs, self._total = offs, total
        self.flat = {name: torch.zeros(max(total, 4), dtype=torch.float32, device=dev) for name in ("param", "grad", "m", "v")}
        self.params, self.grads, self.m, self.v = ({}, {}, {}, {})
        for name, views in (("param", self.params), ("grad", self.grads), ("m", self.m), ("v", self.v)):
            for k in PARAM_KEYS:
                views[k] = self.flat[name][offs[k]:offs[k] + self.n * PARAM_WIDTH[k]]
        for k in PARAM_KEYS:
            self.params[k].copy_(torch.from_numpy(np.ascontiguousarray(params[k], np.float32).reshape(-1)))
        self.proj = binding.Projected(self.n, dev)
        # capacity for the tile intersections: caller's bound, else a generous default
        self.capacity = int(capacity) if capacity is not None else max(1 << 16, 24 * self.n)
        self.bins = binding.Binning(self.capacity, self.K, self.W, self.H, dev)
        self.partials = binding.Partial(self.K, self.W, self.H, dev)
        self.image = torch.empty((self.H, self.W, 3), dtype=torch.float32, device=dev)
        self.T_total = torch.empty((self.H, self.W), dtype=torch.float32, device=dev)
        self.g_image = torch.empty((self.H, self.W, 3), dtype=torch.float32, device=dev)
        self.loss_sum = torch.zeros(1, dtype=torch.float64, device=dev)
        self.pairs = torch.zeros(4, dtype=torch.int64, device=dev)
        self.step_count = 0
        self._cam = None
        self._ws_sort = None
        self._ws_bwd = None

    # -- workspaces are sized per camera resolution (constant here) ----------------------------
    def _workspaces(self, cam):
        if self._ws_sort is None:
            nb = self.ctx.bin_sort_ws_bytes(self.n, self.capacity, self.K, cam)
            self._ws_sort = torch.empty(nb, dtype=torch.uint8, device=self.ctx.device)
            nb = self.ctx.backward_ws_bytes(self.n, self.K, cam)
            self._ws_bwd = torch.empty(nb, dtype=torch.uint8, device=self.ctx.device)

    def forward(self, cam, count_pairs=False):
        """a1-a6: project, bin/sort, render the K partials, compose."""
        self._workspaces(cam)
        self._cam = cam
        c = self.ctx
        c.project(self.params, cam, self.sh_degree, self.proj)
        c.bin_sort(self.proj, self.K, self.part_offsets, cam, self.bins, self._ws_sort)
        c.render_partial(self.proj, self.bins, self.K, cam, self.partials, self.pairs if count_pairs else None)
        c.compose(self.K, self.partials, cam, self.bg, self.image, self.T_total)
        return self.image

    def loss_grad(self, target, scale=1.0):
        """a7: mean-L1 gradient (harness step)."""
        self.ctx.l1_loss_grad(self.image, target, self.g_image, self.loss_sum, scale)

    def backward(self, g_image=None, g_T_total=None, overwrite=False):
        """a8-a10: composition backward, rasteriser backward, projection backward (grads +=, or = for the
        first view of an iteration when overwrite is set)."""
        self.ctx.backward(self.K, self.partials, self._cam, self.bg, self.g_image if g_image is None else g_image,
                          g_T_total, self.params, self.proj, self.bins, self.sh_degree, self.grads, self._ws_bwd,
                          overwrite=overwrite)

    def adam_step(self, n_views=1, zero_grad=False):
        """a11: one Adam step over the flat parameter buffer (five groups = five learning rates, one launch)."""
        self.step_count += 1
        offs = [self._offs[k] for k in PARAM_KEYS] + [self._total]
        self.ctx.adam_groups(self.flat["param"], self.flat["grad"], self.flat["m"], self.flat["v"], offs,
                             [self.lr[k] for k in PARAM_KEYS], step=self.step_count, grad_scale=1.0 / n_views,
                             zero_grad=zero_grad)

    def iteration(self, cams, targets):
        """One training iteration over B views (gradients of the B mean losses are averaged)."""
        for b, (cam, tgt) in enumerate(zip(cams, targets)):
            self.forward(cam)
            self.loss_grad(tgt)
            self.backward(overwrite=(b == 0))     # the first view stores, the others accumulate
        self.adam_step(len(cams))                 # no gradient zeroing needed: next iteration overwrites

    def num_intersections(self) -> int:
        return self.ctx.check_capacity(self.bins)

    def zero_grad(self):
        self.flat["grad"].zero_()
