#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of BASELINE.json on N B200s (replicas only).

A "step" is one pass of the whole hot path over one view of the
workload: project -> bin/sort -> render K partials -> compose -> L1 grad -> compose bwd ->
raster bwd -> project bwd -> Adam.  Workload at N=1: BASELINE.json configs[1] (1M Gaussians, SH3,
1920x1080, K=4 partitions, 2x2 xy grid), synthetic and seeded.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores instead.
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
FLOPS_EVAL = 16      # alpha evaluation of one (pixel, Gaussian) pair: Eq.1 + the skip tests
FLOPS_BLEND_FWD = 12  # one contributing pair in the forward: Eq.3-4 accumulation
FLOPS_BLEND_BWD = 55  # one contributing pair in the backward incl. its 9 reduction adds
FP32_LANES_PER_SM = 128
SM_COUNT = 148
# dram__bytes_read.sum + dram__bytes_write.sum per launch on aerial_1M, from the `ncu --set full` capture summarised in
# profiles/r01e_ncu_full.csv (a profiler number, copied here by hand; null for other workloads)
NCU_TRAFFIC_BYTES = {"aerial_1M": {"k_raster_bwd": 250.9e6, "k_render_fwd": 86.7e6, "adam": 1598.0e6, "project_backward": 520.9e6}}


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
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (profiling recipe)."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-i", str(index), "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
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
        lo, hi = (self.marks + [0, 1e18])[:2] if len(self.marks) >= 2 else (0, 1e18)
        sel = [r for r in rows if lo - 0.05 <= r[0] <= hi + 0.05] or rows
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in sel for i in range(4) if r[3][i].lower().startswith("active")})
        out.update(sm_mhz=statistics.median(r[1] for r in sel), sm_max_mhz=max(r[2] for r in sel), reasons=reasons,
                   samples=len(sel))
        return out


# ------------------------------------------------------------------------------- CPU oracle --
def oracle_sample(sc, n_tiles=96, seed=5):
    """Time the oracle, as it stands, on a bounded sample of the workload: whole-frame stages
    (projection, binning, projection backward) on all N Gaussians, per-pixel stages (render, compose,
    their backwards) on `n_tiles` random tiles, Adam on a 1M-parameter slice; extrapolated to one frame."""
    import oracle
    oracle.build()
    cam = sc.cameras[0]
    camv = cam.as_array()
    W, H = cam.width, cam.height
    TX, TY = (W + 15) // 16, (H + 15) // 16
    rng = np.random.default_rng(seed)
    tiles = np.sort(rng.choice(TX * TY, size=min(n_tiles, TX * TY), replace=False)).astype(np.int32)
    parts = sc.partitions()
    t = {}
    t0 = time.perf_counter()
    proj = [oracle.project(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], sc.sh_degree, camv)
            for p in parts]
    t["project"] = time.perf_counter() - t0
    t0 = time.perf_counter()
    bins = [oracle.bin_sort(pr.means2d, pr.radius, pr.depth, W, H) for pr in proj]
    t["bin_sort"] = time.perf_counter() - t0
    t0 = time.perf_counter()
    pas = [oracle.render_partial(pr.means2d, pr.conic_opacity, pr.rgb, pr.depth, b.vals, b.ranges, W, H,
                                 tile_list=tiles) for pr, b in zip(proj, bins)]
    ct = np.stack([pa.ct for pa in pas]); d = np.stack([pa.d for pa in pas])
    img, Tt, _, _ = oracle.compose(ct, d, sc.bg, tiles)
    _, g_img = oracle.l1(img, sc.targets[0])
    g_ct = oracle.compose_bwd(ct, d, g_img, sc.bg, None, tiles)
    g2 = [oracle.raster_bwd(pr.means2d, pr.conic_opacity, pr.rgb, b.vals, b.ranges, W, H, g_ct[k], tile_list=tiles)
          for k, (pr, b) in enumerate(zip(proj, bins))]
    t["tiles"] = time.perf_counter() - t0
    t0 = time.perf_counter()
    for p, pr, g in zip(parts, proj, g2):
        oracle.project_bwd(p["mean"], p["log_scale"], p["quat"], p["opacity_logit"], p["sh"], sc.sh_degree, camv,
                           pr.radius, pr.clamp, *g)
    t["project_bwd"] = time.perf_counter() - t0
    na = 1_000_000
    pp = np.zeros(na); mm = np.zeros(na); vv = np.zeros(na); gg = rng.standard_normal(na)
    t0 = time.perf_counter()
    oracle.adam(pp, gg, mm, vv, 1e-3, step=1)
    t["adam_1M"] = time.perf_counter() - t0
    frac = len(tiles) / (TX * TY)
    frame_s = t["project"] + t["bin_sort"] + t["project_bwd"] + t["tiles"] / frac + t["adam_1M"] * (59 * sc.N / na)
    walked = sum(pa.walked for pa in pas)
    return dict(frame_s=frame_s, spent_s=sum(t.values()), stages=t, tiles=len(tiles), total_tiles=TX * TY,
                walked_sample=int(walked))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sc = workload(args.workload)
    cam = sc.cameras[0]
    n_tiles = 600
    for _ in range(args.warmup if args.warmup < 2 else 1):
        oracle_sample(sc, n_tiles=8)
    times = []
    for s in range(args.steps):
        times.append(oracle_sample(sc, n_tiles=n_tiles, seed=5 + s))
    frame_s = statistics.mean(x["frame_s"] for x in times)
    mpix = cam.width * cam.height / frame_s / 1e6
    sample = (f"per step: projection/binning/projection-backward on all {sc.N} Gaussians, render+compose+backward on "
              f"{n_tiles} random tiles of {times[0]['total_tiles']} (extrapolated by tile count), Adam on a 1M-parameter "
              f"slice (extrapolated to 59N)")
    line = dict(metric=METRIC, value=mpix, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=frame_s * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", impl="reference",
                config=dict(workload=args.workload, gaussians=sc.N, K=sc.K, width=cam.width, height=cam.height,
                            sh_degree=sc.sh_degree, views_per_step=1),
                cpu_baseline=dict(value=mpix, unit=UNIT, cores=1, kind="oracle", sample=sample),
                e2e=dict(value=mpix, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


# ---------------------------------------------------------------------------------- CUDA path --
def run_ours(args):
    import torch
    from paper_2606_18588_b200 import replicas
    from paper_2606_18588_b200.engine import Trainer

    world, rank, local = replicas.world_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    replicas.init("nccl", local)
    sc = workload(args.workload)
    cam = sc.cameras[0]
    if world > 1:   # every replica trains on its own seeded view of the same scene (weak scaling)
        from paper_2606_18588_b200 import scenes as _sc
        yaw = float(np.random.default_rng(replicas.replica_view_seed(2, rank)).uniform(0, 360))
        if args.workload == "aerial_1M":
            cam = _sc.aerial_camera(cam.width, cam.height, 60.0, 80.0, 45.0, yaw)
    W, H = cam.width, cam.height
    cap = {"aerial_1M": 6_000_000}.get(args.workload)
    tr = Trainer(sc.params, sc.part_offsets, W, H, sc.sh_degree, sc.bg, capacity=cap, device=local)
    c = tr.ctx
    target = torch.from_numpy(sc.targets[0]).cuda()
    tr._workspaces(cam); tr._cam = cam
    K = tr.K
    g_ct = torch.empty((K, H, W, 4), dtype=torch.float32, device="cuda")
    g2d = torch.zeros((tr.n, 12), dtype=torch.float32, device="cuda")
    STAGES = ["project", "bin_sort", "render_partial", "compose", "l1_loss_grad", "compose_backward",
              "raster_backward", "project_backward", "adam"]
    # on the plan path "compose" is the fused kernel compose + L1 + compose backward and the next two stages are empty

    # The step runs under a one-view launch plan (include/splx.h, splx_plan): sparse partial pixels and the
    # geometric visibility state from the partitions' 3-sigma boxes -- both leave every result unchanged
    # (tests/test_gpu_plan.py); --dense times the plain single-view calls instead.
    from paper_2606_18588_b200 import scenes as _scn
    tr.set_aabbs(*_scn.partition_aabbs(sc.params, sc.part_offsets))
    plan, state = tr.bucket_plan([0], [cam], saturation=args.saturation, sparse=True)
    images, T_totals, g_images = tr._view_buffers(1)
    target1 = target[None]

    def step_plan(ev=None):
        def rec(i):
            if ev is not None:
                ev[i].record()
        po = tr.part_offsets
        rec(0); c.project_plan(tr.params, po, plan, tr.sh_degree, tr.proj)
        rec(1); c.bin_sort_plan(tr.proj, po, plan, tr.bins, tr._ws_sort)
        rec(2); c.render_partial_plan(tr.proj, tr.bins, plan, tr.partials)
        rec(3); c.compose_l1_backward_plan(tr.partials, tr.bins, plan, tr.bg, target1, images, T_totals, tr.loss_sum, g_ct,
                                           scale=1.0, sat_eps=args.sat_eps, tile_state_out=state)
        rec(4); rec(5)      # a6 + a7 + a8 run as ONE kernel on this path: stages 4 and 5 are empty
        rec(6); c.raster_backward_plan(tr.proj, tr.bins, plan, tr.partials, g_ct, g2d)
        rec(7); c.project_backward_plan(tr.params, po, plan, tr.sh_degree, tr.proj, g2d, tr.grads, clear_g2d=True,
                                        overwrite=True)
        rec(8); tr.adam_step(1)
        rec(9)

    def step_dense(ev=None):
        def rec(i):
            if ev is not None:
                ev[i].record()
        rec(0); c.project(tr.params, cam, tr.sh_degree, tr.proj)
        rec(1); c.bin_sort(tr.proj, K, tr.part_offsets, cam, tr.bins, tr._ws_sort)
        rec(2); c.render_partial(tr.proj, tr.bins, K, cam, tr.partials)
        rec(3); c.compose(K, tr.partials, cam, tr.bg, tr.image, tr.T_total)
        rec(4); c.l1_loss_grad(tr.image, target, tr.g_image, tr.loss_sum)
        rec(5); c.compose_backward(K, tr.partials, cam, tr.bg, tr.g_image, None, g_ct)
        rec(6); c.raster_backward(tr.proj, tr.bins, K, cam, tr.partials, g_ct, g2d)
        rec(7); c.project_backward(tr.params, cam, tr.sh_degree, tr.proj, g2d, tr.grads, clear_g2d=True, overwrite=True)
        rec(8); tr.adam_step(1)
        rec(9)

    step = step_dense if args.dense else step_plan
    result_image = tr.image if args.dense else images[0]

    def barrier():
        replicas.barrier(cuda=True)

    # unit counts of this view (outside the timed region): pair evaluations and intersections
    tr.pairs.zero_()
    c.project(tr.params, cam, tr.sh_degree, tr.proj)
    c.bin_sort(tr.proj, K, tr.part_offsets, cam, tr.bins, tr._ws_sort)
    c.render_partial(tr.proj, tr.bins, K, cam, tr.partials, tr.pairs)
    M = tr.num_intersections()
    pairs_fwd = int(tr.pairs[0].item())
    pairs_blend = int(tr.pairs[1].item())                          # (pixel, Gaussian) pairs that are blended
    pairs_eval = int(tr.pairs[2].item())                           # alpha evaluations executed after the exact culling
    items_fwd = int(tr.pairs[3].item())                            # (Gaussian, half tile) items that survive the culling
    n_contrib = tr.partials.n_contrib
    pairs_bwd = int(n_contrib.to(torch.int64).sum().item())       # list entries the backward re-evaluates
    n_visible = int((tr.proj.radius > 0).sum().item())
    rng_ = tr.bins.tile_ranges
    live_slots = int((rng_[:, 1] > rng_[:, 0]).sum().item())     # (partition, tile) slots with a non-empty list

    # Every timed pass (eager with stage events, graph replay, end to end) starts from the SAME training state: the
    # parameters and moments are restored first, then W warm-up steps, then K timed steps -- the work of a step
    # drifts as training moves the Gaussians, so passes run one after the other would time different scenes.
    snap = {k: tr.flat[k].clone() for k in ("param", "m", "v")}
    snap_count = tr.step_count

    def restore():
        for k, v in snap.items():
            tr.flat[k].copy_(v)
        tr.step_count = snap_count
        if getattr(tr, "_step_dev", None) is not None:
            tr._step_dev.fill_(snap_count)
        if state is not None:
            pass   # the saturation bytes are rebuilt by the first composition

    sampler = ClockSampler(local) if rank == 0 else None
    restore()
    for _ in range(max(args.warmup, 3)):
        step()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(10)] for _ in range(args.steps)]
    l0 = c.launch_count()
    barrier()
    if sampler: sampler.mark()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for s in range(args.steps):
        step(evs[s])
    e1.record()
    barrier()
    if sampler: sampler.mark()
    launches = c.launch_count() - l0
    ms_total = e0.elapsed_time(e1)
    ms_step = replicas.max_over_ranks(ms_total, cuda=True) / args.steps
    stage_ms = {n: statistics.mean(evs[s][i].elapsed_time(evs[s][i + 1]) for s in range(args.steps))
                for i, n in enumerate(STAGES)}
    clocks = sampler.stop() if sampler else None

    # the same iteration replayed from a CUDA graph (a1-a10 captured once, Adam outside): no per-stage events
    graph_ms = overlap_ms = None
    if not args.dense:
        restore()
        for _ in range(max(args.warmup, 3)):
            tr.step_graph(0, cam, target1, saturation=args.saturation, sat_eps=args.sat_eps)
        barrier()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record()
        for s in range(args.steps):
            tr.step_graph(0, cam, target1, saturation=args.saturation, sat_eps=args.sat_eps)
        g1.record()
        barrier()
        graph_ms = replicas.max_over_ranks(g0.elapsed_time(g1), cuda=True) / args.steps
        # for information (timing.ms_per_step_step_overlapped, never `value`): the same K iterations on the overlapped
        # schedule (Trainer.step_overlapped: the SH group's Adam step and the colour half of the projection on a second
        # stream beside the next geometry half + binning), flush of the last deferred half included.  Measured: no gain --
        # the binning's kernels slow down by as much as the optimiser step takes when they share HBM
        overlap_ms = None
        if not args.no_overlap:
            restore()
            for _ in range(max(args.warmup, 3)):
                tr.step_overlapped(0, cam, target1, saturation=args.saturation, sat_eps=args.sat_eps)
            tr.flush()
            barrier()
            o0, o1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            o0.record()
            for s in range(args.steps):
                tr.step_overlapped(0, cam, target1, saturation=args.saturation, sat_eps=args.sat_eps)
            tr.flush()
            o1.record()
            barrier()
            overlap_ms = replicas.max_over_ranks(o0.elapsed_time(o1), cuda=True) / args.steps

    # end to end through the public API with HOST buffers: the step's input (target image) comes from
    # pinned host memory, the result (rendered image + loss) goes back to pinned host memory, every step
    tgt_host = torch.from_numpy(sc.targets[0]).pin_memory()
    img_host = torch.empty((H, W, 3), dtype=torch.float32).pin_memory()
    loss_host = torch.empty(1, dtype=torch.float64).pin_memory()

    def step_e2e():
        if args.dense:
            target.copy_(tgt_host, non_blocking=True)
            tr.loss_sum.zero_()
            step()
            img_host.copy_(result_image, non_blocking=True)
            loss_host.copy_(tr.loss_sum, non_blocking=True)
            torch.cuda.current_stream().synchronize()
        else:   # the public call: Trainer.step_host (copies on a side stream, overlapped with the kernels)
            tr.step_host(0, cam, tgt_host, img_host, loss_host, saturation=args.saturation, sat_eps=args.sat_eps)

    restore()
    for _ in range(max(args.warmup, 3)):
        step_e2e()
    barrier()
    n_e2e = args.steps
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        step_e2e()
    barrier()
    e2e_ms = replicas.max_over_ranks((time.perf_counter() - t0) * 1e3 / n_e2e, cuda=True)
    if rank != 0:
        replicas.finish()
        return

    pk = peaks()
    # `value`: the iteration as a user runs it (Trainer.step_graph: a1-a10 replayed from a CUDA graph, then Adam), K
    # steps between two events; the eager pass above (10 event records per step) gives the per-stage times
    ms_eager = ms_step
    if graph_ms:
        ms_step = graph_ms
    value_from = ("K steps of Trainer.step_graph (CUDA-graph replay of a1-a10 + Adam)" if graph_ms
                  else "K eager steps with per-stage events")
    if graph_ms and overlap_ms and overlap_ms < graph_ms:
        ms_step = overlap_ms
        value_from = ("K steps of Trainer.step_overlapped + flush (same kernels as step_graph; the SH group's Adam step and "
                      "the colour half of the projection run on a second stream beside the next geometry half + binning)")
    mpix = world * W * H / (ms_step * 1e-3) / 1e6
    # dominant kernel: the rasteriser backward (FP32 issue + shuffles + atomics): algorithmic flops
    dom = max(stage_ms, key=stage_ms.get)
    fp32_peak = SM_COUNT * FP32_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12   # TFLOP/s
    flops_bwd = pairs_bwd * FLOPS_EVAL + pairs_blend * FLOPS_BLEND_BWD
    flops_fwd = pairs_fwd * FLOPS_EVAL + pairs_blend * FLOPS_BLEND_FWD
    hbm_bytes = dict(project=n_visible * 285 + (tr.n - n_visible) * 93, adam=28 * 59 * tr.n,
                     # dense calls: three kernels; plan path: ONE fused kernel (partials once, target in, image + T + g_ct out)
                     compose=(20 * K + 16) * W * H if args.dense else (20 + 16) * 256 * live_slots + (12 + 16) * W * H,
                     compose_backward=(12 + 36 * K) * W * H if args.dense else 0,
                     project_backward=n_visible * 472, l1_loss_grad=36 * W * H if args.dense else 0)
    if dom == "raster_backward":
        ach = flops_bwd / (stage_ms[dom] * 1e-3) / 1e12
        roof = dict(kernel="k_raster_bwd", bound="alu", achieved=ach, peak=fp32_peak, unit="TFLOP/s", frac=ach / fp32_peak,
                    traffic=NCU_TRAFFIC_BYTES.get(args.workload, {}).get("k_raster_bwd"), peak_source=f"148 SMs x 128 FP32 lanes x 2 x {pk['sm_max_mhz']:.0f} MHz ({pk['source']} clock)")
    elif dom == "render_partial":
        ach = flops_fwd / (stage_ms[dom] * 1e-3) / 1e12
        roof = dict(kernel="k_render_fwd", bound="alu", achieved=ach, peak=fp32_peak, unit="TFLOP/s", frac=ach / fp32_peak,
                    traffic=NCU_TRAFFIC_BYTES.get(args.workload, {}).get("k_render_fwd"), peak_source=f"148 SMs x 128 FP32 lanes x 2 x {pk['sm_max_mhz']:.0f} MHz ({pk['source']} clock)")
    else:
        b = hbm_bytes.get(dom, 0)
        ach = b / (stage_ms[dom] * 1e-3) / 1e9
        roof = dict(kernel=dom, bound="hbm", achieved=ach, peak=pk["hbm_gbs"], unit="GB/s", frac=ach / pk["hbm_gbs"],
                    traffic=NCU_TRAFFIC_BYTES.get(args.workload, {}).get(dom), peak_source=pk["source"])
    per_kernel = {}
    for n, b in hbm_bytes.items():
        if b == 0:
            continue
        gbs = b / (stage_ms[n] * 1e-3) / 1e9
        per_kernel[n] = dict(ms=stage_ms[n], algorithmic_GBps=gbs, frac_of_hbm=gbs / pk["hbm_gbs"])
    per_kernel["render_partial"] = dict(ms=stage_ms["render_partial"], Gpairs_per_s=pairs_fwd / stage_ms["render_partial"] / 1e6,
                                        algorithmic_TFLOPs=flops_fwd / stage_ms["render_partial"] / 1e9,
                                        frac_of_fp32=flops_fwd / stage_ms["render_partial"] / 1e9 / fp32_peak)
    per_kernel["raster_backward"] = dict(ms=stage_ms["raster_backward"], Gpairs_per_s=pairs_bwd / stage_ms["raster_backward"] / 1e6,
                                         algorithmic_TFLOPs=flops_bwd / stage_ms["raster_backward"] / 1e9,
                                         frac_of_fp32=flops_bwd / stage_ms["raster_backward"] / 1e9 / fp32_peak)
    per_kernel["bin_sort"] = dict(ms=stage_ms["bin_sort"], intersections=M)

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        o = oracle_sample(sc, n_tiles=1500)
        cpu = dict(value=W * H / o["frame_s"] / 1e6, unit=UNIT, cores=1, kind="oracle",
                   sample=(f"projection/binning/projection-backward on all {sc.N} Gaussians + render/compose/backward on "
                           f"{o['tiles']} random tiles of {o['total_tiles']} (extrapolated by tile count) + Adam on 1M "
                           f"parameters (extrapolated to 59N); {o['spent_s']:.1f} s of CPU work"),
                   ms_per_frame_extrapolated=o["frame_s"] * 1e3)

    line = dict(metric=METRIC, value=mpix, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                ms_per_step=ms_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
                data="synthetic",
                config=dict(workload=args.workload, gaussians=tr.n, K=K, width=W, height=H, sh_degree=sc.sh_degree,
                            views_per_step=1, parallelism=f"replicas x{world} (one GPU per replica, no collective)",
                            path="dense single-view calls" if args.dense else
                                 "one-view launch plan: sparse partials + geometric tile state (results unchanged)",
                            saturation_skipping=bool(args.saturation and not args.dense), live_slots=live_slots,
                            slots=K * ((W + 15) // 16) * ((H + 15) // 16),
                            l2="working set (params+grads+moments 944 MB at 1M) is larger than the 126 MB L2",
                            intersections=M, visible=n_visible, pairs_fwd=pairs_fwd, pairs_bwd=pairs_bwd,
                            pairs_blended=pairs_blend, pairs_evaluated_fwd=pairs_eval, half_tile_items_fwd=items_fwd),
                iters_per_s=world * 1e3 / ms_step, stages_ms=stage_ms, per_kernel=per_kernel, roofline=roof,
                cpu_baseline=cpu, clocks=clocks, gpu_launches=int(launches),
                timing=dict(value_from=value_from, ms_per_step_step_graph=graph_ms, ms_per_step_step_overlapped=overlap_ms,
                            ms_per_step_eager_with_stage_events=ms_eager,
                            stages_ms_from="a separate pass of K eager steps with a CUDA event between stages"),
                e2e=dict(value=world * W * H / (e2e_ms * 1e-3) / 1e6, unit=UNIT, ms_per_step=e2e_ms,
                         h2d_bytes_per_step=int(tgt_host.numel() * 4),
                         d2h_bytes_per_step=int(img_host.numel() * 4 + 8)))
    print(json.dumps(line))
    replicas.finish()


# ------------------------------------------------------- optional subsystems: B views per step --
def run_views(args):
    """`--views B`: one step = one training iteration over B views of the workload (configs[2]-[4] style) through
    Trainer.iteration_views: geometric participants, conflict-free buckets (one launch per stage per bucket),
    saturated-tile skipping.  --no-visibility renders every partition for every view, --no-consolidate runs one
    view per launch, --saturation/--sat-eps as above.  A secondary line: same JSON keys, config.views_per_step = B."""
    import torch
    from paper_2606_18588_b200 import binding, scenes
    from paper_2606_18588_b200.engine import Trainer

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(0)
    sc = workload(args.workload)
    B = min(args.views, len(sc.cameras))
    cams = sc.cameras[:B]
    W, H = cams[0].width, cams[0].height
    cap = {"city_10M": 64_000_000, "street_10M": 200_000_000, "city_40M": 160_000_000,
           "city_100M": 96_000_000}.get(args.workload)
    tr = Trainer(sc.params, sc.part_offsets, W, H, sc.sh_degree, sc.bg, capacity=cap)
    aabbs = scenes.partition_aabbs(sc.params, sc.part_offsets)
    cells = scenes.partition_aabbs(sc.params, sc.part_offsets, inflate_sigma=0.0) if args.cross_filter else None
    sc.params = None                                   # a device-generated scene: release the generator's copy
    torch.cuda.empty_cache()
    tr.sparse_adam = bool(args.sparse_adam)
    if args.no_visibility:   # boxes that contain everything: every partition participates in every view, no tile is invisible
        big = np.float32(1e6)
        tr.set_aabbs(np.full((tr.K, 3), -big), np.full((tr.K, 3), big))
    else:
        tr.set_aabbs(*aabbs)
    cross = None
    if args.cross_filter:    # Q_cross against the cell boxes (boxes of the means); timed once, it is view independent
        tr.set_cross(*cells)
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(); tr.set_cross(*cells); c1.record()
        torch.cuda.synchronize()
        cross = dict(cross_sets_ms=c0.elapsed_time(c1),
                     gaussians_in_Q_cross=int((tr._cross != 0).sum().item()))
    targets = torch.from_numpy(np.stack(sc.targets[:B])).cuda()
    ids = list(range(B))
    kw = dict(consolidate=not args.no_consolidate, saturation=args.saturation, sat_eps=args.sat_eps)
    parts = [tr.participants(v, c) for v, c in zip(ids, cams)]
    groups = tr.buckets(ids, cams, consolidate=not args.no_consolidate)
    sampler = ClockSampler(0)
    for _ in range(max(args.warmup, 3)):
        tr.iteration_views(ids, cams, targets, **kw)
    torch.cuda.synchronize()
    M = tr.num_intersections()
    l0 = tr.ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.mark()
    e0.record()
    for _ in range(args.steps):
        tr.iteration_views(ids, cams, targets, **kw)
    e1.record()
    torch.cuda.synchronize()
    sampler.mark()
    ms = e0.elapsed_time(e1) / args.steps
    launches = tr.ctx.launch_count() - l0
    clocks = sampler.stop()
    skipped = {}
    for key, st in tr._bucket_state.items():
        st = st.cpu().numpy()
        skipped[str(list(key))] = dict(invisible=int((st & binding.TILE_INVISIBLE != 0).sum()),
                                       saturated=int((st & binding.TILE_SATURATED != 0).sum()), slots=int(st.size))
    line = dict(metric=METRIC, value=B * W * H / (ms * 1e-3) / 1e6, unit=UNIT, n_gpus=1, steps=args.steps,
                warmup=max(args.warmup, 3), ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f32", data="synthetic",
                config=dict(workload=args.workload, gaussians=tr.n, K=tr.K, width=W, height=H, sh_degree=sc.sh_degree,
                            views_per_step=B, visibility_prediction=not args.no_visibility,
                            consolidation=not args.no_consolidate, saturation_skipping=bool(args.saturation),
                            optimiser="visible-only Adam (option, not the paper's)" if args.sparse_adam else "dense Adam",
                            cross_boundary_filter=cross, sat_eps=args.sat_eps, participants=[bin(p) for p in parts], buckets=groups,
                            tile_state=skipped, intersections_last_bucket=M,
                            l2="working set (params+grads+moments) is larger than the 126 MB L2"),
                iters_per_s=1e3 / ms, clocks=clocks, gpu_launches=int(launches),
                peak_device_memory_GB=torch.cuda.max_memory_allocated() / 1e9,
                capacity_ok=bool(M <= tr.capacity))
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="aerial_1M")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--dense", action="store_true", help="time the plain single-view calls (dense partial buffers)")
    ap.add_argument("--saturation", action="store_true", help="skip tiles detected as saturated (PAPER.md L231)")
    ap.add_argument("--sat-eps", type=float, default=1e-4)
    ap.add_argument("--views", type=int, default=0, help="B > 0: time iterations over B views (optional subsystems)")
    ap.add_argument("--no-visibility", action="store_true")
    ap.add_argument("--no-consolidate", action="store_true")
    ap.add_argument("--no-overlap", action="store_true", help="do not time the overlapped schedule (Trainer.step_overlapped)")
    ap.add_argument("--cross-filter", action="store_true",
                    help="--views only: cross-boundary per-ray filtering (PAPER.md L474-L476, DESIGN.md s32)")
    ap.add_argument("--sparse-adam", action="store_true",
                    help="--views only: visible-only Adam (an option outside the paper, DESIGN.md s31)")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 2 if args.steps is None else min(args.steps, 4)
        args.warmup = 1 if args.warmup is None else min(args.warmup, 1)
        run_reference(args)
    else:
        args.steps = 50 if args.steps is None else args.steps
        args.warmup = 5 if args.warmup is None else args.warmup
        if args.views > 0:
            args.steps = min(args.steps, 20)
            run_views(args)
        else:
            run_ours(args)


if __name__ == "__main__":
    main()
