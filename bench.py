#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of BASELINE.json on N B200s (replicas only).

A "step" is one training iteration of the workload: for each of its B views the whole hot path (SURVEY.md s8(a) rows
a1..a10: project -> bin/sort -> render K partials -> compose -> L1 grad -> compose bwd -> raster bwd -> project bwd),
then ONE Adam step (a11) -- issued as a single C-ABI call, splx_iteration.  Default workload at N=1: BASELINE.json
configs[4], the largest single-GPU configuration (100M Gaussians, SH3, 1920x1080, K=32 partitions, B=8 views), synthetic
and seeded; `--workload aerial_1M` is configs[1] (B=1), city_10M / city_40M configs[2] / [3].

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

`--impl reference` times the CPU oracle (oracle/, as it stands) on one host core on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fwd+compose+bwd+adam Mpixels/s (train iteration)"
UNIT = "Mpixels/s"

# Algorithmic FP32 work of the blend loops, flops per pair (FMA = 2)
FLOPS_EVAL = 16       # alpha evaluation of one (pixel, Gaussian) pair: Eq.1 + the skip tests
FLOPS_BLEND_FWD = 12  # one contributing pair in the forward: Eq.3-4 accumulation
FLOPS_BLEND_BWD = 55  # one contributing pair in the backward incl. its 9 reduction adds
SM_COUNT, FP32_LANES_PER_SM = 148, 128

#: views per iteration and key capacity of every workload (BASELINE.json configs)
WORKLOADS = {
    "tiny": dict(views=1, capacity=None), "aerial_small": dict(views=1, capacity=None),
    "city_small": dict(views=4, capacity=None), "blocks_small": dict(views=6, capacity=None),
    "aerial_1M": dict(views=1, capacity=6_000_000),
    "city_10M": dict(views=4, capacity=64_000_000), "street_10M": dict(views=4, capacity=200_000_000),
    "city_40M": dict(views=4, capacity=160_000_000), "city_100M": dict(views=8, capacity=96_000_000),
}


def workload(name):
    from paper_2606_18588_b200 import scenes
    if name == "aerial_1M":
        return scenes.aerial()                       # BASELINE configs[1]
    if name == "tiny":
        return scenes.tiny()                         # configs[0]
    if name == "aerial_small":
        return scenes.small_aerial()
    if name == "city_10M":
        return scenes.city()                         # configs[2]: 10M Gaussians, K=8, B=4 views
    if name == "street_10M":                         # the configs[2] scene seen from street level
        return scenes.city(street=True, name="street_10M")
    if name == "city_40M":                           # configs[3]: 40M Gaussians, 1000 m, 4K views, K=16, B=4 (device generator)
        return scenes.city_device(n=40_000_000, width=3840, height=2160, extent=1000.0, n_buildings=800, grid=(4, 4),
                                  altitude=200.0, height_range=(5.0, 60.0), n_views=4, name="city_40M")
    if name == "city_100M":                          # configs[4]: 100M Gaussians, 2000 m, 1080p, K=32, B=8
        return scenes.city_device(n=100_000_000, width=1920, height=1080, extent=2000.0, n_buildings=3200, grid=(8, 4),
                                  altitude=200.0, height_range=(5.0, 80.0), n_views=8, name="city_100M")
    if name == "city_small":
        return scenes.small_city()
    if name == "blocks_small":
        return scenes.small_blocks()
    raise SystemExit(f"unknown workload {name}")


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="MEASURED_PEAKS.json")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback of B200_PROFILING.md (no MEASURED_PEAKS.json)")


def ncu_traffic(workload_name, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu summary of this
    workload (profiles/ncu_traffic.json, written from an `ncu --set full` capture; the file names its source), or None."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(p):
        return None
    try:
        per_kernel = json.load(open(p)).get(workload_name, {})
    except Exception:
        return None
    for name, v in per_kernel.items():      # the file names template instances ("k_adam_groups<1>")
        if name == kernel or name.split("<")[0] == kernel:
            return v
    return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (profiling recipe)."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-i", str(index), "-lms", "20"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None
        self.marks = []

    def mark(self):
        self.marks.append(time.time())

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.p is None:
            return out
        time.sleep(0.12)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = []
        for line in open(self.f.name):
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 8:
                continue
            try:
                ts = time.mktime(time.strptime(parts[0].split(".")[0], "%Y/%m/%d %H:%M:%S")) + float("0." + parts[0].split(".")[1])
                rows.append((ts, float(parts[1]), float(parts[2]), parts[4:8]))
            except Exception:
                continue
        os.unlink(self.f.name)
        if not rows:
            return out
        lo, hi = (self.marks[0], self.marks[-1]) if len(self.marks) >= 2 else (0, 1e18)
        sel = [r for r in rows if lo - 0.05 <= r[0] <= hi + 0.05] or rows
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in sel for i in range(4) if r[3][i].lower().startswith("active")})
        out.update(sm_mhz=statistics.median(r[1] for r in sel), sm_max_mhz=max(r[2] for r in sel), reasons=reasons,
                   samples=len(sel))
        return out


# ------------------------------------------------------------------------------- CPU oracle --
def host_info():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except Exception:
        pass
    return dict(nproc=os.cpu_count(), cpu_model=model)


class PinnedCore:
    """The oracle leg runs pinned to one core (the `taskset -c 0` of SURVEY.md s8(d))."""

    def __enter__(self):
        self.old = None
        try:
            self.old = os.sched_getaffinity(0)
            os.sched_setaffinity(0, {min(self.old)})
        except Exception:
            self.old = None
        return self

    def __exit__(self, *a):
        if self.old is not None:
            try:
                os.sched_setaffinity(0, self.old)
            except Exception:
                pass


def sampled_views(n_views):
    return [0] if n_views == 1 else [0, n_views - 1]          # the first and the last view of the iteration


def oracle_inputs(sc, params, n_views, boxes):
    """What the oracle leg needs, on the host.  The partitions each sampled view renders come from the ORACLE's own
    geometric participants test (oracle.visibility.participants: the conservative regions of reading s21 on the sub-cell boxes of means); of every
    such partition a slice of Gaussians (at most ~4M in total; float64, the oracle's shapes) is copied -- a
    device-generated scene only sends the slices.  params: key -> flat array / tensor over all Gaussians."""
    from oracle import visibility as ov
    from paper_2606_18588_b200 import scenes
    lo, hi, ms, bp = boxes
    cams = [c.as_array() for c in sc.cameras[:n_views]]
    members = {}
    for v in sampled_views(n_views):
        seen = ov.participants(lo, hi, cams[v], ms)      # one bit per BOX
        ks = {int(bp[j]) for j in range(len(bp)) if (seen >> j) & 1}
        members[v] = [k for k in sorted(ks) if sc.part_offsets[k + 1] > sc.part_offsets[k]]
    needed = sorted({k for m in members.values() for k in m})
    n_slice = int(min(1_000_000, max(100_000, 4_000_000 // max(len(needed), 1))))
    parts = {}
    for k in needed:
        a, b = int(sc.part_offsets[k]), int(sc.part_offsets[k + 1])
        b = min(b, a + n_slice)
        p = {}
        for key in scenes.PARAM_KEYS:
            w = scenes.PARAM_WIDTH[key]
            src = params[key]
            v = src.reshape(-1)[w * a:w * b]
            p[key] = (v if isinstance(v, np.ndarray) else v.cpu().numpy()).astype(np.float64)
        p["mean"] = p["mean"].reshape(-1, 3); p["log_scale"] = p["log_scale"].reshape(-1, 3)
        p["quat"] = p["quat"].reshape(-1, 4); p["sh"] = p["sh"].reshape(-1, 16, 3)
        parts[k] = p
    return dict(parts=parts, members=members, part_sizes=[int(sc.part_offsets[k + 1] - sc.part_offsets[k]) for k in range(sc.K)],
                cams=cams, wh=(sc.cameras[0].width, sc.cameras[0].height), targets=sc.targets, sh_degree=sc.sh_degree,
                bg=sc.bg, N=sc.N, K=sc.K, n_slice=n_slice)


def oracle_sample(oi, n_views, budget_s, seed=5):
    """Time the oracle, as it stands, single thread, on a BOUNDED sample of one iteration of the workload and
    extrapolate to the whole iteration.  Per sampled view: projection, binning and projection backward on the slices of
    `oracle_inputs` (scaled to the partition sizes), render + compose + L1 + their backwards on random tiles until the
    time budget is spent (scaled by tile count), Adam on 1M parameters (scaled to 59 N)."""
    import oracle
    oracle.build()
    W, H = oi["wh"]
    TX, TY = (W + 15) // 16, (H + 15) // 16
    rng = np.random.default_rng(seed)
    K = oi["K"]
    t_iter = 0.0
    spent = 0.0
    tiles_done = 0
    walked = 0
    views = sampled_views(n_views)
    per_view_budget = budget_s / len(views)
    for v in views:
        camv = oi["cams"][v]
        mem = oi["members"][v]
        t_whole = 0.0         # stages over whole partitions, scaled from the slices
        proj, bins, scale = {}, {}, {}
        for k in mem:
            p = oi["parts"][k]
            n_k = oi["part_sizes"][k]
            if n_k == 0:
                continue
            sl = p["mean"].shape[0]
            t0 = time.perf_counter()
            pr = oracle.project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], oi["sh_degree"], camv)
            b = oracle.bin_sort(pr.means2d, pr.radius, pr.depth, W, H)
            dt = time.perf_counter() - t0
            proj[k], bins[k], scale[k] = pr, b, n_k / sl
            t_whole += dt * n_k / sl
            spent += dt
        # per-pixel stages on random tiles of the slice scene (lists shortened by the slicing are scaled back below)
        order = rng.permutation(TX * TY).astype(np.int32)
        t_tiles = 0.0
        n_t = 0
        chunk = 4
        while t_tiles < per_view_budget and n_t < TX * TY:
            tiles = np.sort(order[n_t:n_t + chunk])
            t0 = time.perf_counter()
            pas = [oracle.render_partial(proj[k].means2d, proj[k].conic_opacity, proj[k].rgb, proj[k].depth, bins[k].vals,
                                         bins[k].ranges, W, H, tile_list=tiles) for k in proj]
            ct = np.stack([pa.ct for pa in pas]); d = np.stack([pa.d for pa in pas])
            img, Tt, _, _ = oracle.compose(ct, d, oi["bg"], tiles)
            _, g_img = oracle.l1(img, oi["targets"][v])
            g_ct = oracle.compose_bwd(ct, d, g_img, oi["bg"], None, tiles)
            g2 = [oracle.raster_bwd(proj[k].means2d, proj[k].conic_opacity, proj[k].rgb, bins[k].vals, bins[k].ranges, W, H,
                                    g_ct[j], tile_list=tiles) for j, k in enumerate(proj)]
            t_tiles += time.perf_counter() - t0
            walked += sum(pa.walked for pa in pas)
            n_t += len(tiles)
            chunk = min(chunk * 2, 64)
        spent += t_tiles
        tiles_done += n_t
        # projection backward on the slices (zero 2-D gradients cost the same arithmetic)
        t_pb = 0.0
        for k in proj:
            p, pr = oi["parts"][k], proj[k]
            n = pr.radius.shape[0]
            z = lambda w: np.zeros((n, w)) if w > 1 else np.zeros(n)
            t0 = time.perf_counter()
            oracle.project_bwd(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], oi["sh_degree"], camv,
                               pr.radius, pr.clamp, z(2), z(3), z(1), z(3))
            dt = time.perf_counter() - t0
            t_pb += dt * scale[k]
            spent += dt
        # the lists of the slice scene are shorter than the real ones by the slicing ratio; the early exit bounds the walked
        # part of a saturating list, so the tile stages are NOT scaled by the density (if anything a lower bound)
        t_view = t_whole + t_pb + t_tiles * (TX * TY) / max(n_t, 1)
        t_iter += t_view * (n_views / len(views))
    na = 1_000_000
    pp = np.zeros(na); mm = np.zeros(na); vv = np.zeros(na); gg = rng.standard_normal(na)
    t0 = time.perf_counter()
    oracle.adam(pp, gg, mm, vv, 1e-3, step=1)
    dt = time.perf_counter() - t0
    spent += dt
    t_iter += dt * (59 * oi["N"] / na)
    return dict(iter_s=t_iter, spent_s=spent, tiles=tiles_done, total_tiles=TX * TY, views_sampled=views, walked_sample=int(walked))


def oracle_sample_text(o, oi, n_views):
    return (f"one core, oracle as it stands: per sampled view (views {o['views_sampled']} of {n_views}) projection + binning + "
            f"projection backward on slices of <= {oi['n_slice']} Gaussians per rendered partition (scaled to the partition sizes), "
            f"render + compose + L1 + backwards on {o['tiles']} random tiles of {o['total_tiles']} per view of the slice "
            f"scene (scaled by tile count; lists shorter than the full scene's, so a lower bound of the oracle's time), Adam "
            f"on 1M parameters (scaled to 59 N = {59 * oi['N']}); EXTRAPOLATED to the iteration; {o['spent_s']:.1f} s of CPU work")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sc = workload(args.workload)
    B = min(WORKLOADS[args.workload]["views"], len(sc.cameras))
    cam = sc.cameras[0]
    from paper_2606_18588_b200 import scenes
    oi = oracle_inputs(sc, sc.params, B, scenes.partition_boxes(sc.params, sc.part_offsets, sub=args.sub_cells))
    sc.params = None
    total = max(args.steps + args.warmup, 1)
    budget = max(0.3, min(10.0, 120.0 / total))        # tile-stage seconds per step: the whole run ends within minutes
    hi = host_info()
    with PinnedCore():
        for _ in range(args.warmup):
            oracle_sample(oi, B, budget)
        times = [oracle_sample(oi, B, budget, seed=5 + s) for s in range(args.steps)]
    iter_s = statistics.mean(x["iter_s"] for x in times)
    mpix = B * cam.width * cam.height / iter_s / 1e6
    line = dict(metric=METRIC, value=mpix, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=iter_s * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", impl="reference",
                config=dict(workload=args.workload, gaussians=sc.N, K=sc.K, width=cam.width, height=cam.height,
                            sh_degree=sc.sh_degree, views_per_step=B, host=hi),
                cpu_baseline=dict(value=mpix, unit=UNIT, cores=1, kind="oracle", sample=oracle_sample_text(times[0], oi, B),
                                  extrapolated=True, **hi),
                e2e=dict(value=mpix, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


# ---------------------------------------------------------------------------------- CUDA path --
def micro_peaks(ctx, torch):
    """FP32 FMA and MUFU ex2 issue peaks of THIS GPU, measured now (splx_microbench, CUDA events, best of 5)."""
    sink = torch.zeros(1, dtype=torch.float32, device="cuda")
    out = {}
    for kind, name, it in ((0, "fma_tflops", 1 << 14), (1, "ex2_tops", 1 << 12)):
        ctx.microbench(kind, 64, sink)      # warm-up
        best = 0.0
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            work = ctx.microbench(kind, it, sink)
            e1.record()
            torch.cuda.synchronize()
            best = max(best, work / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        out[name] = best
    return out


def run_ours(args):
    import torch
    from paper_2606_18588_b200 import binding, replicas, scenes
    from paper_2606_18588_b200.engine import Trainer

    world, rank, local = replicas.world_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    replicas.init("nccl", local)
    sc = workload(args.workload)
    B = args.views if args.views > 0 else WORKLOADS[args.workload]["views"]
    B = min(B, len(sc.cameras))
    cams = list(sc.cameras[:B])
    if world > 1 and args.workload == "aerial_1M":   # every replica trains on its own seeded view of the same scene (weak scaling)
        yaw = float(np.random.default_rng(replicas.replica_view_seed(2, rank)).uniform(0, 360))
        cams = [scenes.aerial_camera(cams[0].width, cams[0].height, 60.0, 80.0, 45.0, yaw)]
    W, H = cams[0].width, cams[0].height
    tr = Trainer(sc.params, sc.part_offsets, W, H, sc.sh_degree, sc.bg, capacity=WORKLOADS[args.workload]["capacity"], device=local)
    c = tr.ctx
    boxes = scenes.partition_boxes(sc.params, sc.part_offsets, sub=args.sub_cells)
    cells = scenes.partition_boxes(sc.params, sc.part_offsets)[:2] if args.cross_filter else None
    oi = oracle_inputs(sc, tr.params, B, boxes) if (world == 1 and rank == 0 and not args.no_cpu_baseline) else None
    sc.params = None                                   # a device-generated scene: release the generator's copy
    torch.cuda.empty_cache()
    tr.sparse_adam = bool(args.sparse_adam)
    tr.flagged_grads = "always" if args.always_flags else (not args.plain_grads)
    tr.lambda_dssim = float(args.lambda_dssim)
    if args.no_visibility:   # boxes that contain everything: every partition participates in every view, no tile is invisible
        big = np.float32(1e6)
        tr.set_aabbs(np.full((tr.K, 3), -big), np.full((tr.K, 3), big))
    else:                    # boxes of the means + footprint margin: conservative regions (results unchanged)
        tr.set_aabbs(*boxes)
    cross = None
    if args.cross_filter:    # Q_cross against the cell boxes (boxes of the means); view independent
        tr.set_cross(*cells)
        cross = dict(gaussians_in_Q_cross=int((tr._cross != 0).sum().item()))
    ids = list(range(B))
    targets = torch.from_numpy(np.stack(sc.targets[:B])).cuda()
    kw = dict(consolidate=not args.no_consolidate, saturation=args.saturation, sat_eps=args.sat_eps)
    parts = [tr.participants(v, cam) for v, cam in zip(ids, cams)]
    groups = tr.buckets(ids, cams, consolidate=not args.no_consolidate)
    plans = [tr.bucket_plan([ids[i] for i in g], [cams[i] for i in g], args.saturation, True) for g in groups]
    tr._workspaces(cams[0])
    K = tr.K
    ntiles = ((W + 15) // 16) * ((H + 15) // 16)
    single_graph = (B == 1 and not args.no_graph)

    def barrier():
        replicas.barrier(cuda=True)

    # ---- unit counts of this iteration, bucket by bucket (outside the timed regions) -------------------------
    g_ct, g2d = tr.fused_buffers()
    counts = dict(visible=0, participating=0, intersections=0, live_slots=0, pairs_walked_fwd=0, pairs_blended=0,
                  pairs_evaluated_fwd=0, half_tile_items_fwd=0, pairs_walked_bwd=0, dropped_invisible_lists=0)
    per_bucket_M = []
    for (plan, state), grp in zip(plans, groups):
        tr.pairs.zero_()
        tr.forward_plan(plan, count_pairs=True)
        M = tr.num_intersections()
        per_bucket_M.append(M)
        vop = plan.view_of_part
        act = [k for k in range(K) if vop[k] >= 0]
        counts["participating"] += sum(tr.part_offsets[k + 1] - tr.part_offsets[k] for k in act)
        counts["visible"] += int((tr.proj.radius > 0).sum().item()) if len(act) == K else \
            sum(int((tr.proj.radius[tr.part_offsets[k]:tr.part_offsets[k + 1]] > 0).sum().item()) for k in act)
        counts["intersections"] += M
        rg = tr.bins.tile_ranges
        counts["live_slots"] += int((rg[:, 1] > rg[:, 0]).sum().item())
        pw, pb, pe, it = [int(x) for x in tr.pairs.tolist()]
        counts["pairs_walked_fwd"] += pw; counts["pairs_blended"] += pb
        counts["pairs_evaluated_fwd"] += pe; counts["half_tile_items_fwd"] += it
        nc = tr.partials.n_contrib.view(K, -1)
        live_k = (rg.view(K, ntiles, 2)[:, :, 1] > rg.view(K, ntiles, 2)[:, :, 0])
        # entries the backward re-walks: n_contrib of the pixels of live slots (dead slots were never written)
        for k in act:
            if bool(live_k[k].any()):
                pix_live = live_k[k].view((H + 15) // 16, (W + 15) // 16).repeat_interleave(16, 0).repeat_interleave(16, 1)[:H, :W]
                counts["pairs_walked_bwd"] += int(nc[k].view(H, W)[pix_live].to(torch.int64).sum().item())
        counts["dropped_invisible_lists"] += int(tr.bins.num_intersections[1].item())
    if max(per_bucket_M) > tr.capacity:
        raise SystemExit(f"bench.py: {max(per_bucket_M)} intersections exceed the key capacity {tr.capacity}")

    # ---- training state: restored before every timed pass when memory allows (the work of a step drifts as training moves
    # the Gaussians, so passes run one after the other would time different scenes)
    free, _ = torch.cuda.mem_get_info()
    need = 3 * tr.flat["param"].numel() * 4
    can_restore = need < free - (8 << 30)
    snap = {k: tr.flat[k].clone() for k in ("param", "m", "v")} if can_restore else None
    snap_count = tr.step_count

    def restore():
        if snap is not None:
            for k, v in snap.items():
                tr.flat[k].copy_(v)
            tr.step_count = snap_count

    # ---- pass 1: the iteration stage by stage with CUDA events between the stages (per-stage times) ---------------------
    STAGES = ["project", "bin_sort", "render_partial", "compose", "raster_backward", "project_backward", "adam"]
    images, T_totals, g_images = tr._view_buffers(B)

    def staged_iteration(ev):
        """The calls of splx_iteration issued one by one (buckets in order, no pipelining), an event before every stage."""
        po = tr.part_offsets
        if flags:
            tr._touched.zero_()       # (splx_iteration clears the flags with a cudaMemsetAsync)
        for gi, ((plan, state), grp) in enumerate(zip(plans, groups)):
            nb = len(grp)
            tg = targets[grp[0]:grp[0] + 1] if nb == 1 else targets[torch.as_tensor(grp, device="cuda")]
            e = ev[gi]
            # a1 as splx_iteration runs it: the geometry half, the binning, then the colour of the visible list (e[8] between)
            if fused_proj:
                e[0].record(); c.project_plan(tr.params, po, plan, tr.sh_degree, tr.proj)
                e[1].record(); tr._bin_sort(tr.proj, plan, tr.bins, tr._ws_sort)
                e[8].record()
            else:
                e[0].record(); c.project_geometry_plan(tr.params, po, plan, tr.proj)
                e[1].record(); tr._bin_sort(tr.proj, plan, tr.bins, tr._ws_sort)
                e[8].record()
                lst, cnt = c.bin_sort_visible(tr._ws_sort, tr.n, tr.capacity, K, plan.cams[0])
                c.project_colour_list_plan(tr.params, po, plan, tr.sh_degree, tr.proj, lst, cnt)
            e[2].record(); c.render_partial_plan(tr.proj, tr.bins, plan, tr.partials)
            e[3].record()
            if tr.lambda_dssim > 0:
                c.compose_plan(tr.partials, tr.bins, plan, tr.bg, images[:nb], T_totals[:nb], args.sat_eps, state)
                c.dssim_loss_grad(cams[0], images[:nb], tg, g_images[:nb], tr.loss_sum, tr._dssim_ws, tr.lambda_dssim)
                c.compose_backward_plan(tr.partials, tr.bins, plan, tr.bg, g_images[:nb], None, g_ct)
            else:
                c.compose_l1_backward_plan(tr.partials, tr.bins, plan, tr.bg, tg, images[:nb], T_totals[:nb], tr.loss_sum,
                                           g_ct, scale=float(nb), sat_eps=args.sat_eps, tile_state_out=state)
            e[4].record(); c.raster_backward_plan(tr.proj, tr.bins, plan, tr.partials, g_ct, g2d)
            e[5].record()
            if gi == 0 and not flags:
                c.project_backward_plan(tr.params, po, plan, tr.sh_degree, tr.proj, g2d, tr.grads, clear_g2d=True, overwrite=True)
            else:
                if not (flags and (tr.sparse_adam or tr.keep_zero_rows)):     # only the Gaussians that received a 2-D gradient
                    lst, cnt = c.bin_sort_gradient_rows(tr._ws_sort, tr.n, tr.capacity, K, plan.cams[0], g2d)
                else:
                    lst, cnt = c.bin_sort_visible(tr._ws_sort, tr.n, tr.capacity, K, plan.cams[0])
                c.project_backward_list_plan(tr.params, po, plan, tr.sh_degree, tr.proj, g2d, tr.grads, lst, cnt,
                                             clear_g2d=True, touched=tr._touched if flags else None)
            e[6].record()
        tr.adam_step(B, flagged=flags)
        ev[-1][7].record()

    if not single_graph:      # the first iteration over a set of views measures the fraction of Gaussians that receive a gradient
        tr.iteration_views(ids, cams, targets, **kw)
        torch.cuda.synchronize()
        restore()
    flags = tr.flags_decision(ids, plans[0][0]) if not single_graph else tr._use_flags(plans[0][0])
    fused_proj = tr.use_fused_projection([p for p, _ in plans])
    tr._trainset(B, False, flags)     # allocates the D-SSIM workspace / the touched flags
    n_staged = max(3, min(args.steps, 10))
    restore()
    for _ in range(2):
        staged_iteration([[torch.cuda.Event() for _ in range(9)] for _ in plans])
    evs = [[[torch.cuda.Event(enable_timing=True) for _ in range(9)] for _ in plans] for _ in range(n_staged)]
    torch.cuda.synchronize()
    for s in range(n_staged):
        staged_iteration(evs[s])
    torch.cuda.synchronize()
    if flags and not tr.sparse_adam and not tr.keep_zero_rows:
        counts["rows_with_gradient"] = int(tr._touched.sum().item())
    stage_ms = {n: 0.0 for n in STAGES}
    for s in range(n_staged):
        for gi in range(len(plans)):
            e = evs[s][gi]
            for i, n in enumerate(STAGES[:6]):
                stage_ms[n] += e[i].elapsed_time(e[i + 1]) / n_staged
            colour = e[8].elapsed_time(e[2]) / n_staged           # inside [e1, e2): belongs to the projection, not the binning
            stage_ms["project"] += colour
            stage_ms["bin_sort"] -= colour
        stage_ms["adam"] += evs[s][-1][6].elapsed_time(evs[s][-1][7]) / n_staged
    eager_ms = sum(evs[s][0][0].elapsed_time(evs[s][-1][7]) for s in range(n_staged)) / n_staged

    # ---- pass 2 (`value`): K iterations as a user runs them, inputs resident in HBM ----------------------------------------
    def step_value():
        if single_graph:
            tr.step_graph(0, cams[0], targets[0:1], saturation=args.saturation, sat_eps=args.sat_eps)
        else:
            tr.iteration_views(ids, cams, targets, **kw)

    sampler = ClockSampler(local) if rank == 0 else None
    restore()
    l_before = c.launch_count()
    step_value()                                   # (captures the graph of the single-view path)
    torch.cuda.synchronize()
    launches_per_step = c.launch_count() - l_before
    for _ in range(max(args.warmup, 3) - 1):
        step_value()
    barrier()
    if sampler: sampler.mark()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step_value()
    e1.record()
    barrier()
    if sampler: sampler.mark()
    ms_step = replicas.max_over_ranks(e0.elapsed_time(e1), cuda=True) / args.steps
    clocks = sampler.stop() if sampler else None
    tr.check_overflow(wait=True)

    # ---- pass 3 (`e2e`): the same iteration through the C ABI with HOST buffers: the B target images come from pinned host
    # memory and the B rendered images + the loss sums go back to pinned host memory, every step (splx_iteration, SPLX_ITER_HOST)
    tg_host = [torch.from_numpy(sc.targets[i]).pin_memory() for i in ids]
    img_host = [torch.empty((H, W, 3), dtype=torch.float32).pin_memory() for _ in ids]
    loss_host = torch.zeros(2, dtype=torch.float64).pin_memory()

    def step_e2e():
        if single_graph:
            tr.step_host(0, cams[0], tg_host[0], img_host[0], loss_host, saturation=args.saturation, sat_eps=args.sat_eps)
        else:
            tr.iteration_views(ids, cams, tg_host, images_host=img_host, loss_host=loss_host, **kw)
            torch.cuda.current_stream().synchronize()      # the step's result is read on the host

    restore()
    for _ in range(max(args.warmup, 3)):
        step_e2e()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_e2e()
    barrier()
    e2e_ms = replicas.max_over_ranks((time.perf_counter() - t0) * 1e3 / args.steps, cuda=True)
    tr.check_overflow(wait=True)
    loss_l1 = float(loss_host[0]) / (B * W * H * 3)
    if rank != 0:
        replicas.finish()
        return

    # ---- rooflines ---------------------------------------------------------------------------------------------------------
    pk = peaks()
    mp = micro_peaks(c, torch)
    fp32_nominal = SM_COUNT * FP32_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    n_slot_pass = (max(1, (K * ntiles).bit_length()) + 7) // 8
    nv, npart, M = counts["visible"], counts["participating"], counts["intersections"]
    first_overwrite = not flags
    vis0 = nv / max(len(plans), 1)                     # visible Gaussians of an average bucket
    hbm_bytes = dict(
        project=nv * 285 + (npart - nv) * 93,
        bin_sort=4 * npart + 12 * nv + 4 * 16 * nv + 4 * nv + (12 + 24 * n_slot_pass + 8) * M + 8 * K * ntiles * len(plans),
        compose=(20 + 16) * 256 * counts["live_slots"] + (12 + 12 + 4) * W * H * B,
        # flag-tracked rows: every listed Gaussian costs its list entry, radius and 2-D gradient row (56 B); only a row with a
        # non-zero 2-D gradient goes through the kernel (740 B).  rows_with_gradient = flagged Gaussians after the iteration: a
        # LOWER bound of the rows processed (a Gaussian seen by two buckets counts once)
        project_backward=(236 * tr.n + 272 * vis0 + 740 * (nv - vis0)) if first_overwrite else
                         (56 * nv + 740 * counts["rows_with_gradient"] if counts.get("rows_with_gradient") else 740 * nv),
        # flagged gradient rows: 24 B per parameter (param, m, v read + written) + the gradient of the touched rows only
        adam=(24 * 59 * tr.n + tr.n + 4 * 59 * min(counts.get("rows_with_gradient") or nv, tr.n)) if flags else 28 * 59 * tr.n)
    flops_fwd = counts["pairs_walked_fwd"] * FLOPS_EVAL + counts["pairs_blended"] * FLOPS_BLEND_FWD
    flops_bwd = counts["pairs_walked_bwd"] * FLOPS_EVAL + counts["pairs_blended"] * FLOPS_BLEND_BWD
    flops_fwd_exec = counts["pairs_evaluated_fwd"] * FLOPS_EVAL + counts["pairs_blended"] * FLOPS_BLEND_FWD
    per_kernel = {}
    for n, b in hbm_bytes.items():
        gbs = b / (stage_ms[n] * 1e-3) / 1e9
        per_kernel[n] = dict(ms=stage_ms[n], bound="hbm", algorithmic_bytes=int(b), algorithmic_GBps=gbs, frac=gbs / pk["hbm_gbs"])
    per_kernel["compose"]["note"] = ("fused a6+a7+a8; the partials it reads were written by the render kernel just before and are "
                                     "partly L2-resident: the DRAM traffic is below the algorithmic bytes")
    per_kernel["bin_sort"]["note"] = "a chain of ~13 small kernels; latency-bound when the keys fit the 126 MB L2"
    for n, fl, fle in (("render_partial", flops_fwd, flops_fwd_exec), ("raster_backward", flops_bwd, None)):
        t = fl / (stage_ms[n] * 1e-3) / 1e12
        per_kernel[n] = dict(ms=stage_ms[n], bound="alu", algorithmic_TFLOPs=t, frac=t / mp["fma_tflops"],
                             frac_of_nominal_fp32=t / fp32_nominal,
                             unit="walked (pixel, Gaussian) pairs x 16 flop + blended pairs x %d flop" % (FLOPS_BLEND_FWD if n == "render_partial" else FLOPS_BLEND_BWD))
        if fle is not None:     # the exact culling executes only a fraction of the walked pairs
            per_kernel[n]["executed_TFLOPs"] = fle / (stage_ms[n] * 1e-3) / 1e12
            per_kernel[n]["frac_executed_work"] = per_kernel[n]["executed_TFLOPs"] / mp["fma_tflops"]
    if counts["pairs_walked_fwd"]:   # the backward's culling is the forward's: the same executed / walked ratio (it is not counted separately)
        ratio = counts["pairs_evaluated_fwd"] / counts["pairs_walked_fwd"]
        ex = (counts["pairs_walked_bwd"] * ratio * FLOPS_EVAL + counts["pairs_blended"] * FLOPS_BLEND_BWD) / (stage_ms["raster_backward"] * 1e-3) / 1e12
        per_kernel["raster_backward"]["executed_TFLOPs"] = ex
        per_kernel["raster_backward"]["frac_executed_work"] = ex / mp["fma_tflops"]
    dom = max(stage_ms, key=stage_ms.get)
    kname = {"project": "k_project_fwd", "bin_sort": "k_radix_pass", "render_partial": "k_render_fwd", "compose": "k_compose_fused",
             "raster_backward": "k_raster_bwd", "project_backward": "k_project_bwd", "adam": "k_adam_groups"}[dom]
    pkd = per_kernel[dom]
    if pkd["bound"] == "hbm":
        roof = dict(kernel=kname, stage=dom, bound="hbm", achieved=pkd["algorithmic_GBps"], peak=pk["hbm_gbs"], unit="GB/s",
                    frac=pkd["frac"], traffic=ncu_traffic(args.workload, kname), peak_source=pk["source"])
    else:
        roof = dict(kernel=kname, stage=dom, bound="alu", achieved=pkd["algorithmic_TFLOPs"], peak=mp["fma_tflops"], unit="TFLOP/s",
                    frac=pkd["frac"], traffic=ncu_traffic(args.workload, kname),
                    peak_source="FP32 FMA-loop micro-benchmark measured in this run (splx_microbench)")
    roof["share_of_step"] = stage_ms[dom] / sum(stage_ms.values())

    cpu = None
    if oi is not None:
        hi = host_info()
        with PinnedCore():
            o = oracle_sample(oi, B, budget_s=args.cpu_seconds)
        cpu = dict(value=B * W * H / o["iter_s"] / 1e6, unit=UNIT, cores=1, kind="oracle", extrapolated=True,
                   sample=oracle_sample_text(o, oi, B), ms_per_iteration_extrapolated=o["iter_s"] * 1e3, **hi)

    skipped = {}
    for key, st in tr._bucket_state.items():
        st = st.cpu().numpy()
        skipped[str(list(key))] = dict(invisible=int((st & binding.TILE_INVISIBLE != 0).sum()),
                                       saturated=int((st & binding.TILE_SATURATED != 0).sum()), slots=int(st.size))
    mpix = world * B * W * H / (ms_step * 1e-3) / 1e6
    line = dict(metric=METRIC, value=mpix, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                ms_per_step=ms_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
                config=dict(workload=args.workload, gaussians=tr.n, K=K, width=W, height=H, sh_degree=sc.sh_degree, views_per_step=B,
                            parallelism=f"replicas x{world} (one GPU per replica, no collective)",
                            path="splx_iteration: conflict-free buckets under launch plans, sparse partials, conservative geometric "
                                 "tile state (boxes of the means + footprint margin: results unchanged)",
                            visibility_prediction=not args.no_visibility, consolidation=not args.no_consolidate,
                            saturation_skipping=bool(args.saturation), sat_eps=args.sat_eps, lambda_dssim=tr.lambda_dssim,
                            optimiser="visible-only Adam (option, not the paper's)" if args.sparse_adam else "dense Adam",
                            cross_boundary_filter=cross, participants=[bin(p) for p in parts], buckets=groups, tile_state=skipped,
                            slots=K * ntiles * len(plans), l2="working set (params+grads+moments) is larger than the 126 MB L2",
                            unit_counts=counts, intersections_per_bucket=per_bucket_M),
                iters_per_s=world * 1e3 / ms_step, stages_ms=stage_ms, per_kernel=per_kernel, roofline=roof,
                micro_peaks=dict(fma_TFLOPs=mp["fma_tflops"], ex2_Tops=mp["ex2_tops"], nominal_fp32_TFLOPs=fp32_nominal,
                                 how="splx_microbench: 8 independent chains per thread, 8 CTAs x 256 threads per SM, best of 5, CUDA events"),
                cpu_baseline=cpu, clocks=clocks, gpu_launches=int(launches_per_step * args.steps),
                timing=dict(value_from=("K steps of Trainer.step_graph (splx_iteration replayed from a CUDA graph + Adam)" if single_graph
                                        else "K calls of Trainer.iteration_views (one splx_iteration each: all buckets + Adam)"),
                            ms_per_step_eager_stage_by_stage=eager_ms, state_restored_between_passes=bool(can_restore),
                            stages_ms_from=f"a separate pass of {n_staged} iterations issued stage by stage with CUDA events between the stages "
                                           "(buckets one after the other, no pipelining)"),
                loss_l1=loss_l1, peak_device_memory_GB=torch.cuda.max_memory_allocated() / 1e9,
                e2e=dict(value=world * B * W * H / (e2e_ms * 1e-3) / 1e6, unit=UNIT, ms_per_step=e2e_ms,
                         h2d_bytes_per_step=int(B * H * W * 3 * 4), d2h_bytes_per_step=int(B * H * W * 3 * 4 + 16),
                         through="splx_iteration with SPLX_ITER_HOST: pinned host targets in, images + loss sums out, copies on the library's streams"))
    print(json.dumps(line))
    replicas.finish()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="city_100M", choices=sorted(WORKLOADS))
    ap.add_argument("--views", type=int, default=0, help="views per iteration (default: the workload's B)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="tile-stage budget of the oracle leg (cpu_baseline)")
    ap.add_argument("--no-graph", action="store_true", help="B = 1: call splx_iteration every step instead of replaying its CUDA graph")
    ap.add_argument("--saturation", action="store_true", help="skip tiles detected as saturated (PAPER.md L231)")
    ap.add_argument("--sat-eps", type=float, default=1e-4)
    ap.add_argument("--lambda-dssim", type=float, default=0.0, help="weight of the D-SSIM term (PAPER.md L95); 0 = mean L1 only")
    ap.add_argument("--no-visibility", action="store_true")
    ap.add_argument("--sub-cells", type=int, default=8,
                    help="geometric visibility prediction: every partition is covered by sub x sub boxes of means (DESIGN.md s21)")
    ap.add_argument("--no-consolidate", action="store_true")
    ap.add_argument("--cross-filter", action="store_true", help="cross-boundary per-ray filtering (PAPER.md L474-L476, DESIGN.md s32)")
    ap.add_argument("--plain-grads", action="store_true",
                    help="do not track the gradient rows with flags: the first bucket writes every row, Adam reads every row")
    ap.add_argument("--always-flags", action="store_true", help="flag-tracked gradient rows whatever the first bucket covers")
    ap.add_argument("--sparse-adam", action="store_true", help="visible-only Adam (an option outside the paper, DESIGN.md s31)")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 2 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        run_reference(args)
    else:
        args.steps = 20 if args.steps is None else args.steps
        args.warmup = 5 if args.warmup is None else args.warmup
        run_ours(args)


if __name__ == "__main__":
    main()
