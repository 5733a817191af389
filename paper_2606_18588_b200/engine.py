"""Buffer ownership and call sequencing for one training iteration on one B200.

``Trainer`` owns the device memory (parameters, gradients, Adam moments, projected attributes,
binning, partial-pixel buffers) and issues the C-ABI calls of ``include/splx.h`` in the order
of SURVEY.md s3(b).  It performs no arithmetic of the method itself: every step runs in the
CUDA kernels behind ``binding.Context``.  K partitions = K contiguous slices of the SoA.
"""
from __future__ import annotations

import os

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
        self.n = int(params["opacity_logit"].shape[0])
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
        self.loss_sum = torch.zeros(1, dtype=torch.float64, device=dev)
        self.pairs = torch.zeros(4, dtype=torch.int64, device=dev)
        self.step_count = 0
        #: fuse the Adam step into the last projection backward (splx_project_backward_adam_plan).  Off by default:
        #: at 4 CTAs/SM (124 registers) the fused kernel streams the moments at ~4 TB/s, while the stand-alone Adam
        #: kernel runs at 95 % of the HBM roof -- measured 0.44 ms fused against 0.11 + 0.27 ms
        self.fuse_adam = False
        #: accumulating projection backward over the binning's list of visible Gaussians
        #: (splx_project_backward_list_plan) instead of all rows of the participating partitions
        self.use_visible_list = os.environ.get("SPLX_VISIBLE_LIST", "1") == "1"
        #: visible-only ("sparse") Adam -- an OPTION outside the paper: only Gaussians that received a gradient
        #: in the iteration take the step (splx_adam_sparse); no gradient buffer is ever zeroed or overwritten wholesale
        self.sparse_adam = os.environ.get("SPLX_SPARSE_ADAM", "0") == "1"
        self._touched = None
        #: multi-bucket iterations: project + sort of the next bucket on a second stream while this one is blended
        self.pipeline_buckets = os.environ.get("SPLX_PIPELINE", "1") == "1"
        self._cam = None
        self._aabb = None
        self._cross = None          # Q_cross masks (set_cross): cross-boundary filtering on
        self._side = None
        self._ws_sort = None
        self._ws_bwd = None
        # plan path (visibility prediction / consolidated views): buffers with a leading view dimension
        self._images = self._T_totals = self._g_images = None
        self._plan = None
        self._participants = {}     # view id -> partition bitmask (splx_visible_regions)
        self._geom_state = {}       # view id -> host uint8 [K, tiles]
        self._bucket_state = {}     # tuple of view ids -> device uint8 [K * tiles] (geometric | saturated bits)

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

    # ---- launch plans: visibility prediction and consolidated views (L247-L249) ----
    def _view_buffers(self, B):
        if self._images is None or self._images.shape[0] < B:
            dev = self.ctx.device
            self._images = torch.empty((B, self.H, self.W, 3), dtype=torch.float32, device=dev)
            self._T_totals = torch.empty((B, self.H, self.W), dtype=torch.float32, device=dev)
            self._g_images = torch.empty((B, self.H, self.W, 3), dtype=torch.float32, device=dev)
        return self._images[:B], self._T_totals[:B], self._g_images[:B]

    def make_plan(self, cams, view_of_part=None, tile_state=None, sparse=True) -> binding.Plan:
        if view_of_part is None:
            view_of_part = [0] * self.K
        return binding.Plan(cams, view_of_part, tile_state, sparse)

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
        """g_ct [K,H,W,4] and g2d [n,12] of the fused path (g2d starts zeroed and is kept zero by
        splx_project_backward's SPLX_PB_CLEAR_G2D)."""
        if getattr(self, "_g_ct", None) is None:
            dev = self.ctx.device
            self._g_ct = torch.empty((self.K, self.H, self.W, 4), dtype=torch.float32, device=dev)
            self._g2d = torch.zeros((max(self.n, 1), binding.G2D_STRIDE), dtype=torch.float32, device=dev)
        return self._g_ct, self._g2d

    def prepare_adam(self):
        """Host side of the fused optimiser step: count the step.  The bias corrections themselves come from the
        DEVICE-resident counter (splx_adam_bias_step, launched by iteration_fused(adam=True)), so that a captured graph
        advances them at every replay and no host value is read by work that is still in flight."""
        if getattr(self, "_bc_dev", None) is None:
            dev = self.ctx.device
            self._bc_dev = torch.empty(2, dtype=torch.float32, device=dev)
            self._step_dev = torch.full((1,), self.step_count, dtype=torch.int32, device=dev)
        self.step_count += 1

    def _bufs(self, which=0):
        """(projected, binning, sort workspace) set `which`: set 1 is the double buffer of the pipelined multi-bucket
        iteration (the next bucket is projected and binned while the current one is blended)."""
        if which == 0:
            return self.proj, self.bins, self._ws_sort
        if getattr(self, "_alt", None) is None:
            dev = self.ctx.device
            self._alt = (binding.Projected(self.n, dev), binding.Binning(self.capacity, self.K, self.W, self.H, dev),
                         torch.empty_like(self._ws_sort))
        return self._alt

    def _front(self, plan, bufs):
        """a1-a4 of a bucket: project, bin/sort."""
        proj, bins, ws = bufs
        self.ctx.project_plan(self.params, self.part_offsets, plan, self.sh_degree, proj)
        self._bin_sort(proj, plan, bins, ws)

    def _back(self, plan, bufs, targets, overwrite, sat_eps, tile_state_out, adam, n_views):
        """a5-a10 of a bucket: render, fused composition + loss + composition backward, raster and projection backward."""
        proj, bins, ws = bufs
        c = self.ctx
        images, T_totals, _ = self._view_buffers(plan.B)
        g_ct, g2d = self.fused_buffers()
        c.render_partial_plan(proj, bins, plan, self.partials)
        c.compose_l1_backward_plan(self.partials, bins, plan, self.bg, targets, images, T_totals, self.loss_sum, g_ct,
                                   scale=float(plan.B), sat_eps=sat_eps if sat_eps is not None else 0.0,
                                   tile_state_out=tile_state_out)
        c.raster_backward_plan(proj, bins, plan, self.partials, g_ct, g2d)
        if adam:     # the last backward of the iteration takes the optimiser step too (call prepare_adam() first)
            c.adam_bias_step(self._step_dev, self._bc_dev)
            c.project_backward_adam_plan(self.params, self.part_offsets, plan, self.sh_degree, proj, g2d, self.grads,
                                         self.m, self.v, [self.lr[k] for k in PARAM_KEYS], self._bc_dev,
                                         grad_scale=1.0 / n_views, clear_g2d=True, overwrite=overwrite)
        elif self.sparse_adam:    # every launch walks the visible list; the flags say which rows to store and which to add to
            if self._touched is None:
                self._touched = torch.zeros(max(self.n, 1), dtype=torch.uint8, device=self.ctx.device)
            lst, cnt = c.bin_sort_visible(ws, self.n, self.capacity, self.K, plan.cams[0])
            c.project_backward_list_plan(self.params, self.part_offsets, plan, self.sh_degree, proj, g2d, self.grads,
                                         lst, cnt, clear_g2d=True, touched=self._touched)
        elif not overwrite and self.use_visible_list:   # an accumulating launch over the binning's visible list only
            lst, cnt = c.bin_sort_visible(ws, self.n, self.capacity, self.K, plan.cams[0])
            c.project_backward_list_plan(self.params, self.part_offsets, plan, self.sh_degree, proj, g2d, self.grads,
                                         lst, cnt, clear_g2d=True)
        else:
            c.project_backward_plan(self.params, self.part_offsets, plan, self.sh_degree, proj, g2d, self.grads,
                                    clear_g2d=True, overwrite=overwrite)
        return images

    def iteration_fused(self, plan: binding.Plan, targets, overwrite=True, sat_eps=None, tile_state_out=None, adam=False,
                        n_views=1):
        """a1-a10 under a plan with composition, mean-L1 loss and composition backward in ONE kernel
        (splx_compose_l1_backward_plan) -- the training path; the staged calls remain for stage-wise parity.
        targets: device [B,H,W,3].  Returns images[B,H,W,3]."""
        self._workspaces(plan.cams[0])
        self._plan = plan
        bufs = self._bufs(0)
        self._front(plan, bufs)
        return self._back(plan, bufs, targets, overwrite, sat_eps, tile_state_out, adam, n_views)

    def loss_grad_plan(self, targets):
        """a7 for B views at once: targets[B,H,W,3]; every view's loss is its own mean (scale = B)."""
        B = self._plan.B
        images, _, g_images = self._view_buffers(B)
        self.ctx.l1_loss_grad(images, targets, g_images, self.loss_sum, float(B))

    def backward_plan(self, overwrite=False, g_images=None):
        plan = self._plan
        _, _, gi = self._view_buffers(plan.B)
        self.ctx.backward_plan(self.part_offsets, plan, self.partials, self.bg, gi if g_images is None else g_images,
                               None, self.params, self.proj, self.bins, self.sh_degree, self.grads, self._ws_bwd,
                               overwrite=overwrite)

    def set_cross(self, cell_lo, cell_hi, support_sigma=3.0):
        """Cross-boundary per-ray filtering (L474-L476) on: Q_cross of every Gaussian against the cell
        boxes (to be called again when the Gaussians change); the depth intervals and Omega come from set_aabbs.
        cell_lo=None switches it off."""
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
        if getattr(plan, "_zr", None) is None:
            plan._zr = binding.cross_depth_ranges(self._aabb[0], self._aabb[1], plan)
        self.ctx.bin_sort_filtered_plan(proj, self.part_offsets, plan, self._cross, plan._zr, bins, ws)

    def set_aabbs(self, lo, hi):
        """Static partition boxes (scenes.partition_aabbs) for the geometric visibility prediction."""
        self._aabb = (np.ascontiguousarray(lo, np.float32), np.ascontiguousarray(hi, np.float32))
        self._participants.clear(); self._geom_state.clear(); self._bucket_state.clear()

    def participants(self, view_id, cam) -> int:
        """GetParticipants(v) (L249): partitions whose box meets the view frustum; cached per view id."""
        if view_id not in self._participants:
            state, part = binding.visible_regions(self._aabb[0], self._aabb[1], cam)
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
        state = self._bucket_state[key]
        return self.make_plan(cams, vop, state, sparse), (state if saturation else None)

    def iteration_views(self, view_ids, cams, targets, consolidate=True, saturation=True, sat_eps=1e-4, sparse=True):
        """One training iteration over B views with visibility prediction: geometric participants and tile
        regions, saturated tiles skipped from the previous visit of the same bucket on, conflict-free views
        consolidated into one launch per stage.  targets: device tensor [B,H,W,3].  Returns the number of launches
        of the forward (= buckets)."""
        groups = self.buckets(view_ids, cams, consolidate)
        if self.fuse_adam:
            self.prepare_adam()
        G = len(groups)
        plans = [self.bucket_plan([view_ids[i] for i in grp], [cams[i] for i in grp], saturation, sparse) for grp in groups]
        tgs = [targets[grp[0]:grp[0] + 1] if len(grp) == 1 else targets[torch.as_tensor(grp, device=targets.device)]
               for grp in groups]
        self._workspaces(cams[0])
        if G == 1 or not self.pipeline_buckets:
            for gi in range(G):
                self.iteration_fused(plans[gi][0], tgs[gi], overwrite=(gi == 0), sat_eps=sat_eps, tile_state_out=plans[gi][1],
                                     adam=(self.fuse_adam and gi == G - 1), n_views=len(view_ids))
        else:
            # Two streams, double-buffered projected / binning sets: bucket g+1 is projected and sorted (latency-bound
            # kernels that leave most of the SMs idle) on the side stream while bucket g is blended on the main one.
            dev = self.ctx.device
            main = torch.cuda.current_stream(dev)
            if getattr(self, "_front_stream", None) is None:
                self._front_stream = torch.cuda.Stream(dev)
            side = self._front_stream
            ev_front = [torch.cuda.Event() for _ in range(G)]
            ev_back = [torch.cuda.Event() for _ in range(G)]
            side.wait_stream(main)                       # the parameters of the previous optimiser step
            self.ctx.set_stream(side.cuda_stream)
            self._front(plans[0][0], self._bufs(0))
            ev_front[0].record(side)
            self.ctx.set_stream(main.cuda_stream)
            for gi in range(G):
                if gi + 1 < G:
                    if gi >= 1:
                        side.wait_event(ev_back[gi - 1])  # buffer set (gi + 1) % 2 was last read by the back half of gi - 1
                    self.ctx.set_stream(side.cuda_stream)
                    self._front(plans[gi + 1][0], self._bufs((gi + 1) % 2))
                    ev_front[gi + 1].record(side)
                    self.ctx.set_stream(main.cuda_stream)
                main.wait_event(ev_front[gi])
                self._plan = plans[gi][0]
                self._back(plans[gi][0], self._bufs(gi % 2), tgs[gi], gi == 0, sat_eps, plans[gi][1],
                           self.fuse_adam and gi == G - 1, len(view_ids))
                ev_back[gi].record(main)
            side.wait_stream(main)
        if self.sparse_adam:
            self.step_count += 1
            self.ctx.adam_sparse(self.params, self.grads, self.m, self.v, self._touched, [self.lr[k] for k in PARAM_KEYS],
                                 step=self.step_count, grad_scale=1.0 / len(view_ids))
        elif not self.fuse_adam:
            self.adam_step(len(view_ids))
        return len(groups)

    # ---- end to end from HOST buffers ---------------------------------------------------------------
    def _host_body(self, main, side, plan, state, target_host, image_host, loss_host, sat_eps):
        """a1-a10 with the host copies on the side stream: the target travels while the forward renders (it is
        first needed by the loss), the image travels while the backward runs."""
        side.wait_stream(main)
        with torch.cuda.stream(side):
            self._target_dev[0].copy_(target_host, non_blocking=True)
            self._ev_target.record(side)
        self.loss_sum.zero_()
        self._workspaces(plan.cams[0])
        self._plan = plan
        c = self.ctx
        images, T_totals, _ = self._view_buffers(1)
        g_ct, g2d = self.fused_buffers()
        c.project_plan(self.params, self.part_offsets, plan, self.sh_degree, self.proj)
        self._bin_sort(self.proj, plan, self.bins, self._ws_sort)
        c.render_partial_plan(self.proj, self.bins, plan, self.partials)
        main.wait_event(self._ev_target)            # the target is first needed by the fused composition + loss
        c.compose_l1_backward_plan(self.partials, self.bins, plan, self.bg, self._target_dev, images, T_totals,
                                   self.loss_sum, g_ct, scale=1.0, sat_eps=sat_eps, tile_state_out=state)
        if image_host is not None:
            side.wait_stream(main)
            with torch.cuda.stream(side):
                image_host.copy_(images[0], non_blocking=True)
        c.raster_backward_plan(self.proj, self.bins, plan, self.partials, g_ct, g2d)
        if self.fuse_adam:
            c.adam_bias_step(self._step_dev, self._bc_dev)
            c.project_backward_adam_plan(self.params, self.part_offsets, plan, self.sh_degree, self.proj, g2d, self.grads,
                                         self.m, self.v, [self.lr[k] for k in PARAM_KEYS], self._bc_dev, grad_scale=1.0,
                                         clear_g2d=True, overwrite=True)
        else:
            c.project_backward_plan(self.params, self.part_offsets, plan, self.sh_degree, self.proj, g2d, self.grads,
                                    clear_g2d=True, overwrite=True)
        main.wait_stream(side)
        if loss_host is not None:    # after the image has left: the two copies share one device-to-host engine, and
            loss_host.copy_(self.loss_sum, non_blocking=True)   # 8 bytes queued behind 25 MB would stall this stream

    def step_host(self, view_id, cam, target_host, image_host=None, loss_host=None, saturation=False, sat_eps=1e-4,
                  graph=True):
        """One whole training iteration (a1-a11) on one view whose target image lives in pinned HOST memory; the
        rendered image and the loss go back to pinned host memory.  With graph=True the launches of a1-a10 and the
        copies are captured once per (view, buffers) into a CUDA graph and replayed (one launch per step instead of
        ~20); the Adam step is fused into the projection backward, its bias corrections travel through a pinned
        host pair that the graph's copy node reads at replay time.  Returns after the device has drained, so the host
        buffers are valid."""
        dev = self.ctx.device
        main = torch.cuda.current_stream(dev)
        if self.fuse_adam:
            self.prepare_adam()
        if self._side is None:
            self._side = torch.cuda.Stream(dev)
        if getattr(self, "_graphs", None) is None:
            self._ev_target = torch.cuda.Event()
            self._target_dev = torch.empty((1, self.H, self.W, 3), dtype=torch.float32, device=dev)
            self._graphs = {}
        if not graph:
            plan, state = (self.bucket_plan([view_id], [cam], saturation=saturation) if self._aabb is not None
                           else (self.make_plan([cam]), None))
            self._host_body(main, self._side, plan, state, target_host, image_host, loss_host, sat_eps)
        else:
            key = (view_id, target_host.data_ptr(), image_host.data_ptr() if image_host is not None else 0,
                   loss_host.data_ptr() if loss_host is not None else 0, bool(saturation), float(sat_eps), self.fuse_adam)
            if key not in self._graphs:
                plan, state = (self.bucket_plan([view_id], [cam], saturation=saturation) if self._aabb is not None
                               else (self.make_plan([cam]), None))
                self._workspaces(cam)
                self._view_buffers(1)
                self.fused_buffers()
                torch.cuda.synchronize(dev)
                g = torch.cuda.CUDAGraph()
                old = main.cuda_stream
                with torch.cuda.graph(g):
                    cap = torch.cuda.current_stream(dev)
                    self.ctx.set_stream(cap.cuda_stream)
                    try:
                        self._host_body(cap, self._side, plan, state, target_host, image_host, loss_host, sat_eps)
                    finally:
                        self.ctx.set_stream(old)
                self._graphs[key] = (g, plan)          # the plan owns the host arrays the capture read
            self._graphs[key][0].replay()
        if not self.fuse_adam:
            self.adam_step(1)        # outside the graph: its bias correction is a launch argument
        main.synchronize()

    # ---- the same iteration, scheduled so that HBM-bound and latency-bound stages overlap ----------------------
    def _adam_part(self, sh: bool, step: int, n_views=1):
        """Adam (a11) on the SH group only, or on the four geometry groups (mean, log_scale, quat, opacity) only."""
        o = self._offs
        if sh:
            a, b = o["sh"], self._total
            offs, lrs = [0, b - a], [self.lr["sh"]]
        else:
            a, b = 0, o["sh"]
            keys = [k for k in PARAM_KEYS if k != "sh"]
            offs, lrs = [o[k] for k in keys] + [b], [self.lr[k] for k in keys]
        f = self.flat
        self.ctx.adam_groups(f["param"][a:b], f["grad"][a:b], f["m"][a:b], f["v"][a:b], offs, lrs, step=step,
                             grad_scale=1.0 / n_views)

    def step_overlapped(self, view_id, cam, target_dev, saturation=False, sat_eps=1e-4):
        """step_graph with the same kernels and the same arithmetic on a different schedule.  Two facts are used:
        the binning needs only the GEOMETRY half of the projection (which reads 11 of a Gaussian's 59 parameters),
        and the SH colour is not needed before the blend.  So the Adam step of the SH group -- 81 % of the
        optimiser's bytes, bound by HBM -- is deferred to a second stream where it runs, followed by the colour half
        of the next iteration's projection, beside that iteration's geometry half and binning (a chain of small,
        latency-bound kernels that leaves the memory system idle).  Parameters are complete only after flush()."""
        assert not self.fuse_adam and not self.sparse_adam
        dev = self.ctx.device
        c = self.ctx
        main = torch.cuda.current_stream(dev)
        if self._side is None:
            self._side = torch.cuda.Stream(dev)
        side = self._side
        if getattr(self, "_ographs", None) is None:
            self._ographs = {}
            self._pending_sh = 0          # step number whose SH half of Adam has not run yet (0 = none)
            self._ev = [torch.cuda.Event() for _ in range(3)]
        key = (view_id, target_dev.data_ptr(), bool(saturation), float(sat_eps))
        if key not in self._ographs:
            plan, state = (self.bucket_plan([view_id], [cam], saturation=saturation) if self._aabb is not None
                           else (self.make_plan([cam]), None))
            self._workspaces(cam)
            self._view_buffers(1)
            self.fused_buffers()
            bufs = self._bufs(0)
            torch.cuda.synchronize(dev)
            graphs = []
            for body in (lambda: self._bin_sort(self.proj, plan, self.bins, self._ws_sort),
                         lambda: (self.loss_sum.zero_(), self._back(plan, bufs, target_dev, True, sat_eps, state, False, 1))):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    c.set_stream(torch.cuda.current_stream(dev).cuda_stream)
                    try:
                        body()
                    finally:
                        c.set_stream(main.cuda_stream)
                graphs.append(g)
            self._ographs[key] = (graphs[0], graphs[1], plan)
        g_sort, g_back, plan = self._ographs[key]
        self._plan = plan
        ev_bwd, ev_geom, ev_col = self._ev
        # main: geometry half (its parameters are final: the geometry groups were stepped on this stream)
        c.project_parts_plan(self.params, self.part_offsets, plan, self.sh_degree, self.proj, binding.PROJECT_GEOMETRY)
        ev_geom.record(main)
        # side: SH half of the previous step's Adam (after that step's backward), then the colour half
        c.set_stream(side.cuda_stream)
        try:
            if self._pending_sh:
                side.wait_event(ev_bwd)
                self._adam_part(True, self._pending_sh)
                self._pending_sh = 0
            side.wait_event(ev_geom)
            c.project_parts_plan(self.params, self.part_offsets, plan, self.sh_degree, self.proj, binding.PROJECT_COLOUR)
            ev_col.record(side)
        finally:
            c.set_stream(main.cuda_stream)
        g_sort.replay()                     # a2-a4 beside the side stream's work
        main.wait_event(ev_col)
        g_back.replay()                     # a5-a10
        ev_bwd.record(main)
        self.step_count += 1
        self._adam_part(False, self.step_count)
        self._pending_sh = self.step_count

    def flush(self):
        """Run what step_overlapped deferred: afterwards every parameter has taken every step."""
        if getattr(self, "_pending_sh", 0):
            main = torch.cuda.current_stream(self.ctx.device)
            main.wait_event(self._ev[0])
            self._adam_part(True, self._pending_sh)
            self._pending_sh = 0

    def step_graph(self, view_id, cam, target_dev, saturation=False, sat_eps=1e-4):
        """One whole training iteration on one view with the target already on the device ([1,H,W,3]): a1-a10
        replayed from a CUDA graph captured at the first call for this (view, target), then Adam.  Asynchronous."""
        dev = self.ctx.device
        if self.fuse_adam:
            self.prepare_adam()           # this step's bias corrections (the captured copy node reads them at replay)
        if getattr(self, "_dgraphs", None) is None:
            self._dgraphs = {}
        key = (view_id, target_dev.data_ptr(), bool(saturation), float(sat_eps), self.fuse_adam)
        if key not in self._dgraphs:
            plan, state = (self.bucket_plan([view_id], [cam], saturation=saturation) if self._aabb is not None
                           else (self.make_plan([cam]), None))
            self._workspaces(cam)
            self._view_buffers(1)
            self.fused_buffers()
            main = torch.cuda.current_stream(dev)
            torch.cuda.synchronize(dev)
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                self.ctx.set_stream(torch.cuda.current_stream(dev).cuda_stream)
                try:
                    self.loss_sum.zero_()
                    self.iteration_fused(plan, target_dev, overwrite=True, sat_eps=sat_eps, tile_state_out=state,
                                         adam=self.fuse_adam)
                finally:
                    self.ctx.set_stream(main.cuda_stream)
            self._dgraphs[key] = (g, plan)
        self._dgraphs[key][0].replay()
        if not self.fuse_adam:
            self.adam_step(1)            # outside the graph: its bias correction is a launch argument
