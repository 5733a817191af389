"""Buffer ownership for training on one B200: ``Trainer`` owns the device memory (parameters, gradients, Adam
moments, projected attributes, binning, partial-pixel buffers) and hands it to the C ABI of ``include/splx.h``.

A whole training iteration -- a1-a10 for every bucket of views, the optimiser step, the host copies of the
end-to-end path -- is ONE library call (``splx_iteration``, csrc/iteration.cu); this module only fills in its structs.
The stage-by-stage methods (``forward``, ``loss_grad``, ``backward``, ``forward_plan`` ...) issue the single-stage calls
in the order of SURVEY.md s3(b) and exist for stage-wise parity tests.  No arithmetic of the method happens here.
K partitions = K contiguous slices of the SoA.
"""
from __future__ import annotations

import ctypes as C

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


class CapacityError(RuntimeError):
    """A bucket had more tile intersections than ``Trainer.capacity``: its farthest keys were dropped."""


class Trainer:
    def __init__(self, params: dict, part_offsets, width, height, sh_degree=3, bg=(0.0, 0.0, 0.0),
                 capacity=None, device=0, cfg=None, lr=None, max_views=binding.MAX_VIEWS):
        self.ctx = binding.Context(device, cfg=cfg)
        self.cfg = cfg
        dev = self.ctx.device
        self.n = int(params["opacity_logit"].shape[0])
        self.K = len(part_offsets) - 1
        self.part_offsets = [int(x) for x in part_offsets]
        self._po = (C.c_int64 * (self.K + 1))(*self.part_offsets)
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
            src = params[k]
            if isinstance(src, torch.Tensor):       # a device-generated scene (scenes.city_device)
                self.params[k].copy_(src.reshape(-1))
            else:
                self.params[k].copy_(torch.from_numpy(np.ascontiguousarray(src, np.float32).reshape(-1)))
        self.proj = binding.Projected(self.n, dev)
        # capacity for the tile intersections: caller's bound, else a generous default
        self.capacity = int(capacity) if capacity is not None else max(1 << 16, 24 * self.n)
        self.bins = binding.Binning(self.capacity, self.K, self.W, self.H, dev)
        self.partials = binding.Partial(self.K, self.W, self.H, dev)
        self.image = torch.empty((self.H, self.W, 3), dtype=torch.float32, device=dev)
        self.T_total = torch.empty((self.H, self.W), dtype=torch.float32, device=dev)
        self.g_image = torch.empty((self.H, self.W, 3), dtype=torch.float32, device=dev)
        self.loss_sum = torch.zeros(2, dtype=torch.float64, device=dev)      # [0] sum |image - target|, [1] sum SSIM
        self.pairs = torch.zeros(4, dtype=torch.int64, device=dev)
        self.step_count = 0
        self.max_views = int(max_views)
        #: weight of the D-SSIM term of PAPER.md L95 (L = L_RGB + lambda L_D-SSIM; 0 = mean L1 only, the harness loss of
        #: BASELINE.json configs[0]; DESIGN.md s33 takes lambda = 0.2 when it is switched on)
        self.lambda_dssim = 0.0
        #: visible-only ("sparse") Adam -- an OPTION outside the paper: only Gaussians that received a gradient
        #: in the iteration take the step (splx_adam_sparse); no gradient buffer is ever zeroed or overwritten wholesale
        self.sparse_adam = False
        #: the training path tracks the gradient rows an iteration reaches with one flag byte per Gaussian (splx_trainset.touched):
        #: rows no view saw are neither zeroed, written nor read -- at 100M Gaussians a view sees ~2 % of them -- and the dense
        #: Adam step takes their gradient as zero (splx_adam_groups_flagged: same result as the plain buffer)
        self.flagged_grads = True
        #: multi-bucket iterations: project + sort of the next bucket on a second stream while this one is blended
        self.pipeline_buckets = True
        #: a visible Gaussian that no pixel blended has a zero gradient: the projection backward of splx_iteration runs over the
        #: Gaussians that received a 2-D gradient only (splx_bin_sort_gradient_rows; same result: an unflagged row counts as
        #: zero, adding zero changes nothing).  True keeps every visible row (SPLX_ITER_KEEP_ZERO_ROWS); the visible-only
        #: optimiser option always keeps them
        self.keep_zero_rows = False
        #: a1 inside splx_iteration: None = fused (one kernel) when every partition takes part in every bucket -- then most
        #: Gaussians are visible (aerial views) --, else geometry -> binning -> colour of the visible list (city views, where
        #: most participating Gaussians are culled); True / False force one or the other.  Same results bit for bit
        self.fused_projection = None
        self._touched = None
        self._cam = None
        self._aabb = None           # (lo, hi, max_scale or None): boxes of the geometric visibility prediction
        self._cross = None          # Q_cross masks (set_cross): cross-boundary filtering on
        self._ws_sort = None
        self._ws_bwd = None
        self._alt = None
        self._images = None
        self._plan = None
        self._participants = {}     # view id -> partition bitmask (splx_visible_regions)
        self._geom_state = {}       # view id -> host uint8 [K, tiles]
        self._bucket_state = {}     # tuple of view ids -> device uint8 [K * tiles] (geometric | saturated bits)
        self._bucket_open = {}      # tuple of view ids -> number of slots without the INVISIBLE bit (conservative regions), else 0
        self._bucket_map = {}       # tuple of view ids -> device numbering of those slots (splx_slot_map)
        self._row_fraction = {}     # tuple of view ids of an iteration -> fraction of the Gaussians that received a gradient
        self._part_max_scale = None
        self._graphs = {}
        self._m_host = torch.zeros(max(self.max_views, 1), dtype=torch.int64).pin_memory()   # M of every bucket
        self._m_event = None
        self._m_buckets = 0

    # -- workspaces are sized per camera resolution (constant here) ----------------------------
    def _workspaces(self, cam):
        if self._ws_sort is None:
            nb = self.ctx.bin_sort_ws_bytes(self.n, self.capacity, self.K, cam)
            self._ws_sort = torch.empty(nb, dtype=torch.uint8, device=self.ctx.device)
            nb = self.ctx.backward_ws_bytes(self.n, self.K, cam)
            self._ws_bwd = torch.empty(nb, dtype=torch.uint8, device=self.ctx.device)

    # ---- stage by stage (parity surface) ---------------------------------------------------------------------
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

    def adam_step(self, n_views=1, zero_grad=False, flagged=False):
        """a11: one Adam step over the flat parameter buffer (five groups = five learning rates, one launch).  flagged: the
        gradient rows are tracked by the `touched` flags of the last splx_iteration (untouched rows count as zero)."""
        self.step_count += 1
        offs = [self._offs[k] for k in PARAM_KEYS] + [self._total]
        lrs = [self.lr[k] for k in PARAM_KEYS]
        f = self.flat
        if self.sparse_adam and flagged:
            self.ctx.adam_sparse(self.params, self.grads, self.m, self.v, self._touched, lrs, step=self.step_count,
                                 grad_scale=1.0 / n_views)
        elif flagged:
            self.ctx.adam_groups_flagged(f["param"], f["grad"], f["m"], f["v"], offs, [PARAM_WIDTH[k] for k in PARAM_KEYS], self.n,
                                         self._touched, lrs, step=self.step_count, grad_scale=1.0 / n_views)
        else:
            self.ctx.adam_groups(f["param"], f["grad"], f["m"], f["v"], offs, lrs, step=self.step_count,
                                 grad_scale=1.0 / n_views, zero_grad=zero_grad)

    def iteration(self, cams, targets):
        """One training iteration over B views through the single-stage calls (gradients of the B mean losses are averaged)."""
        for b, (cam, tgt) in enumerate(zip(cams, targets)):
            self.forward(cam)
            self.loss_grad(tgt)
            self.backward(overwrite=(b == 0))     # the first view stores, the others accumulate
        self.adam_step(len(cams))                 # no gradient zeroing needed: next iteration overwrites

    def num_intersections(self) -> int:
        return self.ctx.check_capacity(self.bins)

    def zero_grad(self):
        self.flat["grad"].zero_()

    # ---- launch plans: visibility prediction and consolidated views (L247-L249) ----
    def _view_buffers(self, B):
        if self._images is None or self._images.shape[0] < B:
            dev = self.ctx.device
            nb = max(B, self.max_views)
            self._images = torch.empty((nb, self.H, self.W, 3), dtype=torch.float32, device=dev)
            self._T_totals = torch.empty((nb, self.H, self.W), dtype=torch.float32, device=dev)
            self._g_images = torch.empty((nb, self.H, self.W, 3), dtype=torch.float32, device=dev)
            self._graphs.clear()
        return self._images[:B], self._T_totals[:B], self._g_images[:B]

    def make_plan(self, cams, view_of_part=None, tile_state=None, sparse=True, open_slots=0, slot_map=None) -> binding.Plan:
        """open_slots != 0 (splx_plan.open_slots): the numbering of the open slots is built here (splx_slot_map, one small
        launch) unless the caller passes the one it keeps for these (tile_state, view_of_part, open_slots)."""
        if view_of_part is None:
            view_of_part = [0] * self.K
        ms = getattr(self, "_part_max_scale", None)
        if open_slots and slot_map is None:
            slot_map = self.ctx.slot_map(binding.Plan(cams, view_of_part, tile_state, sparse, ms, open_slots))
        return binding.Plan(cams, view_of_part, tile_state, sparse, ms, open_slots, slot_map)

    def forward_plan(self, plan: binding.Plan, sat_eps=None, tile_state_out=None, count_pairs=False):
        """a1-a6 for all views of the plan in one launch per stage; returns images[B,H,W,3]."""
        self._workspaces(plan.cams[0])
        self._plan = plan
        c = self.ctx
        images, T_totals, _ = self._view_buffers(plan.B)
        c.project_plan(self.params, self.part_offsets, plan, self.sh_degree, self.proj)
        self._bin_sort(self.proj, plan, self.bins, self._ws_sort)
        c.render_partial_plan(self.proj, self.bins, plan, self.partials, self.pairs if count_pairs else None)
        c.compose_plan(self.partials, self.bins, plan, self.bg, images, T_totals,
                       sat_eps if sat_eps is not None else 0.0, tile_state_out)
        return images

    def fused_buffers(self):
        """g_ct [K,H,W,4] and g2d [n,12] of the training path (g2d starts zeroed and is kept zero by
        splx_project_backward's SPLX_PB_CLEAR_G2D)."""
        if getattr(self, "_g_ct", None) is None:
            dev = self.ctx.device
            self._g_ct = torch.empty((self.K, self.H, self.W, 4), dtype=torch.float32, device=dev)
            self._g2d = torch.zeros((max(self.n, 1), binding.G2D_STRIDE), dtype=torch.float32, device=dev)
        return self._g_ct, self._g2d

    def loss_grad_plan(self, targets):
        """a7 for B views at once: targets[B,H,W,3]; every view's loss is its own mean (scale = B)."""
        B = self._plan.B
        images, _, g_images = self._view_buffers(B)
        self.ctx.l1_loss_grad(images[:B], targets, g_images[:B], self.loss_sum, float(B))

    def backward_plan(self, overwrite=False, g_images=None):
        plan = self._plan
        _, _, gi = self._view_buffers(plan.B)
        self.ctx.backward_plan(self.part_offsets, plan, self.partials, self.bg, gi[:plan.B] if g_images is None else g_images,
                               None, self.params, self.proj, self.bins, self.sh_degree, self.grads, self._ws_bwd,
                               overwrite=overwrite)

    def set_cross(self, cell_lo, cell_hi, support_sigma=3.0):
        """Cross-boundary per-ray filtering (L474-L476) on: Q_cross of every Gaussian against the cell
        boxes (to be called again when the Gaussians change); the depth intervals and Omega come from set_aabbs.
        cell_lo=None switches it off."""
        self._graphs.clear()
        if cell_lo is None:
            self._cross = None
            return
        if self._cross is None:
            self._cross = torch.empty(self.n, dtype=torch.int64, device=self.ctx.device)
        self.ctx.cross_sets(self.params, self.part_offsets, cell_lo, cell_hi, self._cross, support_sigma)

    def _bin_sort(self, proj, plan, bins, ws):
        if self._cross is None:
            self.ctx.bin_sort_plan(proj, self.part_offsets, plan, bins, ws)
            return
        self.ctx.bin_sort_filtered_plan(proj, self.part_offsets, plan, self._cross, self._depth_ranges(plan), bins, ws)

    def _depth_ranges(self, plan):
        if getattr(plan, "_zr", None) is None:
            plan._zr = np.ascontiguousarray(binding.cross_depth_ranges(self._part_box[0], self._part_box[1], plan), np.float32)
        return plan._zr

    def set_aabbs(self, lo, hi, max_scale=None, box_part=None):
        """Static boxes for the geometric visibility prediction (L212).  With max_scale (scenes.partition_boxes) the boxes
        are boxes of MEANS covering the partitions (box j belongs to partition box_part[j]; None = one box per partition)
        and splx_visible_regions builds the conservative regions of reading s21: no list the binning builds is cut --
        the training path.  Without max_scale the boxes are taken as they are (tests of
        the region geometry itself, e.g. the 3-sigma boxes of scenes.partition_aabbs)."""
        lo = np.ascontiguousarray(lo, np.float32).reshape(-1, 3)
        hi = np.ascontiguousarray(hi, np.float32).reshape(-1, 3)
        bp = None if box_part is None else np.ascontiguousarray(box_part, np.int32)
        assert bp is not None or lo.shape[0] == self.K, "one box per partition, or box_part"
        self._aabb = (lo, hi, None if max_scale is None else np.ascontiguousarray(max_scale, np.float32), bp)
        # one box per partition (the union of its boxes): the depth intervals D^k of the cross-boundary filter (s32)
        plo = np.full((self.K, 3), np.inf, np.float32); phi = np.full((self.K, 3), -np.inf, np.float32)
        for j in range(lo.shape[0]):
            k = j if bp is None else int(bp[j])
            plo[k] = np.minimum(plo[k], lo[j]); phi[k] = np.maximum(phi[k], hi[j])
        empty = ~np.isfinite(plo).all(1)
        plo[empty] = 0; phi[empty] = 0
        self._part_box = (plo, phi)
        # the largest scale of every partition: splx_plan.max_scale (the projection's reach test on the mean alone)
        self._part_max_scale = None
        if max_scale is not None:
            pms = np.zeros(self.K, np.float32)
            for j in range(lo.shape[0]):
                k = j if bp is None else int(bp[j])
                pms[k] = max(pms[k], float(self._aabb[2][j]))
            self._part_max_scale = pms
        self._participants.clear(); self._geom_state.clear(); self._bucket_state.clear(); self._bucket_open.clear(); self._bucket_map.clear(); self._graphs.clear()

    def participants(self, view_id, cam) -> int:
        """GetParticipants(v) (L249): partitions whose boxes meet the view frustum; cached per view id."""
        if view_id not in self._participants:
            lo, hi, ms, bp = self._aabb
            state, part = binding.visible_regions(lo, hi, cam, ms, bp, self.K, self.cfg)
            for k in range(self.K):                       # an empty partition never participates
                if self.part_offsets[k + 1] == self.part_offsets[k]:
                    part &= ~(1 << k)
                    state[k] = binding.TILE_INVISIBLE
            self._participants[view_id] = part
            self._geom_state[view_id] = state
        return self._participants[view_id]

    def buckets(self, view_ids, cams, consolidate=True, max_views=binding.MAX_VIEWS):
        """Conflict-free buckets (L249) over the given views: list of lists of positions into view_ids."""
        parts = [self.participants(v, c) for v, c in zip(view_ids, cams)]
        if not consolidate:
            return [[i] for i in range(len(view_ids))]
        bucket_of, nb = binding.schedule_views(parts, max_views)
        out = [[] for _ in range(nb)]
        for i, b in enumerate(bucket_of):
            out[b].append(i)
        return out

    def bucket_plan(self, view_ids, cams, saturation=True, sparse=True):
        """Plan of one conflict-free bucket: every partition renders the view it participates in; the tile state
        (geometric bits now, saturated bits as compose detects them) persists per bucket across iterations."""
        key = tuple(view_ids)
        vop = [-1] * self.K
        for j, (v, cam) in enumerate(zip(view_ids, cams)):
            part = self.participants(v, cam)
            for k in range(self.K):
                if (part >> k) & 1:
                    assert vop[k] < 0, "views of a bucket must not share a partition"
                    vop[k] = j
        if key not in self._bucket_state:
            st = np.full((self.K, self._geom_state[view_ids[0]].shape[1]), binding.TILE_INVISIBLE, np.uint8)
            for k in range(self.K):
                if vop[k] >= 0:
                    st[k] = self._geom_state[view_ids[vop[k]]][k]
            self._bucket_state[key] = torch.from_numpy(st.reshape(-1)).to(self.ctx.device)
            # conservative regions (boxes of means + max_scale, reading s21): an INVISIBLE slot holds no intersection, so
            # the slot sort may renumber the open ones (splx_plan.open_slots); the geometric bits never change afterwards
            self._bucket_open[key] = int((st & binding.TILE_INVISIBLE == 0).sum()) if self._part_max_scale is not None else 0
        state = self._bucket_state[key]
        n_open = self._bucket_open.get(key, 0)
        if n_open and key not in self._bucket_map:         # built once per bucket: the INVISIBLE bits never change
            self._bucket_map[key] = self.ctx.slot_map(binding.Plan(cams, vop, state, sparse, self._part_max_scale, n_open))
        return self.make_plan(cams, vop, state, sparse, n_open, self._bucket_map.get(key)), (state if saturation else None)

    # ---- one library call per iteration (splx_iteration) -------------------------------------------------------
    def _frontset(self, which):
        proj, bins, ws = (self.proj, self.bins, self._ws_sort) if which == 0 else self._alt
        return binding.FrontsetS(proj.struct(), bins.struct(), ws.data_ptr(), ws.numel())

    def _trainset(self, n_views, pipelined, flags=False):
        """splx_trainset over this trainer's buffers (allocating the ones the training path needs on first use)."""
        dev = self.ctx.device
        self._view_buffers(max(n_views, 1))
        g_ct, g2d = self.fused_buffers()
        if getattr(self, "_targets_dev", None) is None or self._targets_dev.shape[0] < self._images.shape[0]:
            self._targets_dev = torch.empty_like(self._images)
        if pipelined and self._alt is None:
            self._alt = (binding.Projected(self.n, dev), binding.Binning(self.capacity, self.K, self.W, self.H, dev),
                         torch.empty_like(self._ws_sort))
        if self.lambda_dssim > 0 and getattr(self, "_dssim_ws", None) is None:
            nf = self.ctx.dssim_ws_floats(self.W, self.H)
            self._dssim_ws = torch.empty(binding.MAX_VIEWS * nf, dtype=torch.float32, device=dev)
        flags = flags or self.sparse_adam
        if flags and self._touched is None:
            self._touched = torch.zeros(max(self.n, 1), dtype=torch.uint8, device=dev)
        ts = binding.TrainsetS()
        ts.params = binding.gaussians_struct(self.params)
        ts.grads = binding.gaussians_struct(self.grads)
        ts.K = self.K
        ts.part_offsets = C.cast(self._po, C.c_void_p)
        ts.sh_degree = self.sh_degree
        ts.bg[:] = [float(x) for x in self.bg]
        ts.front[0] = self._frontset(0)
        if pipelined:
            ts.front[1] = self._frontset(1)
        ts.partials = self.partials.struct()
        ts.g_ct, ts.g2d = g_ct.data_ptr(), g2d.data_ptr()
        ts.images, ts.T_totals, ts.g_images = self._images.data_ptr(), self._T_totals.data_ptr(), self._g_images.data_ptr()
        ts.targets = self._targets_dev.data_ptr()
        ts.dssim_ws = self._dssim_ws.data_ptr() if self.lambda_dssim > 0 else None
        ts.loss_sum = self.loss_sum.data_ptr()
        ts.max_views = self._images.shape[0]
        ts.cross_mask = self._cross.data_ptr() if self._cross is not None else None
        ts.touched = self._touched.data_ptr() if flags else None
        return ts

    def _adam_cfg(self, step):
        offs = (C.c_int64 * 6)(*([self._offs[k] for k in PARAM_KEYS] + [self._total]))
        lrs = (C.c_float * 5)(*[float(self.lr[k]) for k in PARAM_KEYS])
        wds = (C.c_int32 * 5)(*[PARAM_WIDTH[k] for k in PARAM_KEYS])
        f = self.flat
        a = binding.AdamCfgS(f["param"].data_ptr(), f["grad"].data_ptr(), f["m"].data_ptr(), f["v"].data_ptr(), 5,
                             C.cast(offs, C.c_void_p), C.cast(lrs, C.c_void_p), 0.9, 0.999, 1e-15, int(step),
                             C.cast(wds, C.c_void_p), 1 if self.sparse_adam else 0,
                             binding.gaussians_struct(self.m), binding.gaussians_struct(self.v))
        a._keep = (offs, lrs, wds)
        return a

    def _bucket_structs(self, plans, groups):
        """ctypes array of splx_bucket for the plans [(binding.Plan, state_out or None)] over the view positions `groups`."""
        arr = (binding.BucketS * len(plans))()
        keep = []
        for i, ((plan, state_out), grp) in enumerate(zip(plans, groups)):
            vi = (C.c_int32 * len(grp))(*[int(x) for x in grp])
            zr = self._depth_ranges(plan) if self._cross is not None else None
            arr[i].plan = plan._s
            arr[i].view_index = C.cast(vi, C.c_void_p)
            arr[i].tile_state_out = state_out.data_ptr() if state_out is not None else None
            arr[i].part_depth_range = zr.ctypes.data if zr is not None else None
            keep += [vi, zr, plan]
        arr._keep = keep
        return arr

    def check_overflow(self, wait=False):
        """Raise CapacityError if a bucket of the last iteration overflowed the key capacity (its count M comes back through
        a pinned host mirror written by splx_iteration; read only once the device has passed that point)."""
        if self._m_event is None:
            return
        if wait:
            self._m_event.synchronize()
        if self._m_event.query():
            m = int(self._m_host[:self._m_buckets].max())
            self._m_event = None
            if m > self.capacity:
                raise CapacityError(f"{m} tile intersections exceed the capacity {self.capacity}: the farthest keys were dropped")

    def use_fused_projection(self, plans) -> bool:
        if self.fused_projection is not None:
            return bool(self.fused_projection)
        return all(v >= 0 for p in plans for v in p.view_of_part)

    def _run_iteration(self, plans, groups, n_views, targets, sat_eps, adam=True, host=False, images_out=None,
                       loss_out=None, flags=False):
        """plans: [(Plan, state_out)], groups: view positions per plan; targets: list of raw pointers per view."""
        if not torch.cuda.is_current_stream_capturing():
            self.check_overflow()
        self._workspaces(plans[0][0].cams[0])
        pipelined = self.pipeline_buckets and len(plans) > 1
        ts = self._trainset(n_views, pipelined, flags)
        bk = self._bucket_structs(plans, groups)
        cfg = None
        if adam:
            self.step_count += 1
            cfg = self._adam_cfg(self.step_count)
        self._plan = plans[-1][0]
        self.ctx.iteration(ts, bk, n_views, targets, images_out, loss_out, self._m_host.data_ptr(), host=host,
                           sat_eps=0.0 if sat_eps is None else sat_eps, lambda_dssim=self.lambda_dssim, adam=cfg,
                           fused_projection=self.use_fused_projection([p for p, _ in plans]),
                           keep_zero_rows=self.sparse_adam or self.keep_zero_rows)   # (Adam may run outside the call)
        self._m_buckets = len(plans)
        return ts, bk

    def iteration_fused(self, plan: binding.Plan, targets, overwrite=True, sat_eps=None, tile_state_out=None):
        """a1-a10 of ONE bucket under a plan (no optimiser step).  targets: device [B,H,W,3].  Returns images[B,H,W,3]."""
        assert overwrite, "a single bucket always stores its gradient"
        B = plan.B
        hw3 = self.H * self.W * 3 * 4
        self._run_iteration([(plan, tile_state_out)], [list(range(B))], B, [targets.data_ptr() + b * hw3 for b in range(B)],
                            sat_eps, adam=False)
        return self._images[:B]

    def iteration_views(self, view_ids, cams, targets, consolidate=True, saturation=True, sat_eps=1e-4, sparse=True,
                        images_host=None, loss_host=None):
        """One training iteration over B views with visibility prediction: geometric participants and tile regions,
        saturated tiles skipped from the previous visit of the same bucket on, conflict-free views consolidated into one
        launch per stage, then Adam -- all inside splx_iteration.  targets: device tensor [B,H,W,3], or a list of B
        PINNED HOST tensors [H,W,3] (then images_host: list of pinned host tensors or None, loss_host: pinned double[2]
        or None receive the results: the end-to-end path).  Returns the number of buckets."""
        groups = self.buckets(view_ids, cams, consolidate)
        plans = [self.bucket_plan([view_ids[i] for i in grp], [cams[i] for i in grp], saturation, sparse) for grp in groups]
        B = len(view_ids)
        host = not isinstance(targets, torch.Tensor)
        if host:
            tptr = [t.data_ptr() for t in targets]
            iptr = [t.data_ptr() for t in images_host] if images_host is not None else None
            lptr = loss_host.data_ptr() if loss_host is not None else None
        else:
            hw3 = self.H * self.W * 3 * 4
            tptr, iptr, lptr = [targets.data_ptr() + b * hw3 for b in range(B)], None, None
        # flag-tracked gradient rows also pay when the first bucket covers most partitions but few Gaussians RECEIVE a gradient
        # (street-level views: 15.3 -> 14.5 ms; aerial views, where nearly every Gaussian does: 1.61 -> 1.69 ms): the first
        # iteration over a set of views runs with flags and measures that fraction (one synchronisation, once)
        key = tuple(view_ids)
        probe = self.flagged_grads is True and not self.sparse_adam and key not in self._row_fraction
        flags = True if probe else self.flags_decision(view_ids, plans[0][0])
        self._run_iteration(plans, groups, B, tptr, sat_eps, adam=True, host=host, images_out=iptr, loss_out=lptr, flags=flags)
        if probe and not self.keep_zero_rows and not torch.cuda.is_current_stream_capturing():
            self._row_fraction[key] = float(self._touched.sum().item()) / max(self.n, 1)
        self._m_event = torch.cuda.Event()
        self._m_event.record(torch.cuda.current_stream(self.ctx.device))
        return len(groups)

    def flags_decision(self, view_ids, first_plan) -> bool:
        """Flag-tracked gradient rows for an iteration over these views?  The static rule of _use_flags, or the measured
        fraction of Gaussians that receive a gradient (known after the first iteration over them) below 30 %."""
        return self._use_flags(first_plan) or self._row_fraction.get(tuple(view_ids), 1.0) < 0.3

    def _use_flags(self, first_plan):
        """Track the gradient rows with flags (splx_trainset.touched) when that saves work: when the first bucket's
        partitions hold most of the Gaussians it writes nearly every row anyway and the plain '=' pass is the cheaper one
        (measured on aerial_1M and city_10M, where every view sees every partition)."""
        if self.sparse_adam:
            return True
        if not self.flagged_grads:
            return False
        if self.flagged_grads == "always":
            return True
        held = sum(self.part_offsets[k + 1] - self.part_offsets[k] for k, v in enumerate(first_plan.view_of_part) if v >= 0)
        return held < 0.75 * self.n

    # ---- one view per iteration, replayed from a CUDA graph -----------------------------------------------------
    def _single_view_plan(self, view_id, cam, saturation):
        if self._aabb is not None:
            return self.bucket_plan([view_id], [cam], saturation=saturation)
        return self.make_plan([cam]), None

    def _graph_step(self, key, plan, state, target_ptr, sat_eps, host, image_ptr, loss_ptr):
        """a1-a10 of one view captured once into a CUDA graph and replayed (one launch per step instead of ~20), then Adam
        outside the graph (its step number is a launch argument)."""
        dev = self.ctx.device
        if key not in self._graphs:
            main = torch.cuda.current_stream(dev)
            self._workspaces(plan.cams[0])
            flags = self._use_flags(plan)
            self._trainset(1, False, flags)
            torch.cuda.synchronize(dev)
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                self.ctx.set_stream(torch.cuda.current_stream(dev).cuda_stream)
                try:
                    keep = self._run_iteration([(plan, state)], [[0]], 1, [target_ptr], sat_eps, adam=False, host=host,
                                               images_out=[image_ptr] if image_ptr else None, loss_out=loss_ptr,
                                               flags=flags)
                finally:
                    self.ctx.set_stream(main.cuda_stream)
            self._graphs[key] = (g, plan, keep, flags)
        self._graphs[key][0].replay()
        self.adam_step(1, flagged=self._graphs[key][3])

    def step_graph(self, view_id, cam, target_dev, saturation=False, sat_eps=1e-4):
        """One whole training iteration on one view with the target already on the device ([1,H,W,3]).  Asynchronous."""
        key = ("dev", view_id, target_dev.data_ptr(), bool(saturation), float(sat_eps), self.lambda_dssim)
        plan, state = (None, None) if key in self._graphs else self._single_view_plan(view_id, cam, saturation)
        self._graph_step(key, plan, state, target_dev.data_ptr(), sat_eps, False, None, None)

    def step_host(self, view_id, cam, target_host, image_host=None, loss_host=None, saturation=False, sat_eps=1e-4,
                  graph=True):
        """One whole training iteration (a1-a11) on one view whose target image lives in PINNED HOST memory; the rendered
        image and the loss sums (double[2]) go back to pinned host memory.  The copies run inside splx_iteration on the
        library's own streams beside the kernels.  Returns after the device has drained: the host buffers are valid."""
        dev = self.ctx.device
        iptr = image_host.data_ptr() if image_host is not None else None
        lptr = loss_host.data_ptr() if loss_host is not None else None
        if graph:
            key = ("host", view_id, target_host.data_ptr(), iptr, lptr, bool(saturation), float(sat_eps), self.lambda_dssim)
            plan, state = (None, None) if key in self._graphs else self._single_view_plan(view_id, cam, saturation)
            self._graph_step(key, plan, state, target_host.data_ptr(), sat_eps, True, iptr, lptr)
        else:
            plan, state = self._single_view_plan(view_id, cam, saturation)
            self._run_iteration([(plan, state)], [[0]], 1, [target_host.data_ptr()], sat_eps, adam=True, host=True,
                                images_out=[iptr] if iptr else None, loss_out=lptr, flags=self._use_flags(plan))
        torch.cuda.current_stream(dev).synchronize()
        m = int(self._m_host[0])
        if m > self.capacity:
            raise CapacityError(f"{m} tile intersections exceed the capacity {self.capacity}: the farthest keys were dropped")
