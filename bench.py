#!/usr/bin/env python
"""bench.py -- fwd+bwd megapixels/s of the tile-based splatting hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--view 0]

A "step" is one pass of the whole hot path over one view: xpr_project -> xpr_bin_sort ->
xpr_rasterize_fwd -> (L1 loss gradient, torch) -> xpr_rasterize_bwd -> xpr_project_bwd.
Workload: BASELINE.json configs[2] ("3DGS unbounded-scene scale": 1,000,000 Gaussians, 1920x1080),
the configuration BASELINE.json:north_star quotes its target on.  Synthetic seeded scene.
Multi-GPU: replicas only; each rank runs the same step, no data-path collective.
One JSON line on stdout (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC, UNIT = "fwd_bwd_megapixels_per_s", "MP/s"
WORKLOADS = {1: "configs[0] tiny 3DGS 1k Gaussians 64x64", 2: "configs[1] 3DGS object-scale 100k Gaussians 800x800",
             3: "configs[2] 3DGS unbounded-scene 1M Gaussians 1920x1080",
             4: "configs[3] 3DGUT fisheye 1M Gaussians 1920x1080", 5: "configs[4] 3DGS stress 3M Gaussians 1920x1080"}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--view", type=int, default=0)
    ap.add_argument("--views", type=int, default=1,
                    help="V > 1: a step renders the batch of views view .. view+V-1 of the scene with ONE call per stage "
                         "(xpr_config.views; SURVEY 8(f) f3; meant for --config 5, whose scene has four views); the metric "
                         "counts the pixels of all V images")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--no-plain", action="store_true", help="skip the extra timing of the plain path (tile_cull 0)")
    ap.add_argument("--tile-cull", type=int, default=1, choices=(0, 1),
                    help="1: binning with the paper's tile_cull (XPR-3DGS, PAPER L149/L268-281; same image); "
                         "0: rectangle overlap only")
    ap.add_argument("--tile-order", type=int, default=-1, choices=(-1, 0, 1),
                    help="1: compositing kernels walk the tiles longest list first (xpr_config.tile_order; scheduling "
                         "only); -1: the pipeline's default (on for 64 <= tiles < 4096)")
    ap.add_argument("--fuse-loss", type=int, default=1, choices=(0, 1),
                    help="1: the loss gradient is formed inside the compositing backward (xpr_rasterize_bwd_loss) instead of a "
                         "separate xpr_loss_grad pass (colour pass of the 2D evaluation only; same results)")
    ap.add_argument("--overlap-fill", type=int, default=-1, choices=(-1, 0, 1, 2, 4),
                    help="pipeline option overlap_fill: the zero-fill of the parameter gradients on a second stream, forked at the "
                         "forward compositing kernel (4), the compositing backward (1) or the binning stage (2); 0: inside "
                         "xpr_project_bwd; -1 the pipeline's default (4)")
    ap.add_argument("--features", type=int, default=0, choices=(0, 1),
                    help="1: also render the depth image and the accumulated opacity and take their gradients "
                         "(SURVEY 8(f) f3, DESIGN.md 6.8; with --ray-eval 1 through the ray kernels; not part of the headline workload)")
    ap.add_argument("--featn", type=int, default=0,
                    help="C > 0: after the timed steps, also time xpr_rasterize_featn_fwd / _bwd with C seeded feature "
                         "channels on the lists of the last step (reported as 'featn'; not part of the step)")
    ap.add_argument("--ray-eval", type=int, default=0, choices=(0, 1),
                    help="1: XPR-3DGUT evaluation along the pixel ray (SURVEY 8(f) f2; meant for --config 4) instead of "
                         "the 2D conic of north_star")
    ap.add_argument("--linprim", type=float, default=0.0,
                    help="M > 0: time XPR-LinPrim instead (SURVEY 8(f) f4, DESIGN.md 11): one forward + backward step on the "
                         "config's scene read as octahedra with half-axes = M x the Gaussian scales (DESIGN.md uses 3); "
                         "one GPU, pinhole configs (1, 2, 3, 5)")
    ap.add_argument("--sort-compare", action="store_true",
                    help="after the timed steps, also time cub::DeviceRadixSort::SortPairs (libxpr_cubcmp.so, built on demand; "
                         "never on the path) on the same (key, value) pairs in emission order, beside xpr_bin_sort "
                         "(reported as 'cub_compare'; BASELINE.json:north_star)")
    ap.add_argument("--stages", action="store_true", help="also print per-stage times to stderr")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def rank_env():
    """(world, rank, local_rank) from the torchrun environment; (1, 0, 0) when launched plainly."""
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def max_over_ranks(value_ms: float, world: int, device):
    """Replicas only: the job's time is the slowest rank's.  One all-reduce(MAX) of a scalar."""
    if world <= 1:
        return float(value_ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value_ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world: int, megapixels: float, ms_per_step: float) -> float:
    """Whole-job MP/s of `world` replicas that each render `megapixels` per step in `ms_per_step` (max over ranks)."""
    return world * megapixels / (ms_per_step / 1e3)


def oracle_step(xo, scenes, sc, view, np, tile_cull=0, ray_eval=0, features=0, views=1):
    """One fwd+bwd step of the CPU oracle, as it stands (never tuned); a batch of views is a loop over the views."""
    t_all, pairs = 0.0, 0
    for v in range(view, view + max(1, views)):
        dt, n = _oracle_view(xo, scenes, sc, v, np, tile_cull, ray_eval, features)
        t_all += dt; pairs += n
    return t_all, pairs


def _oracle_view(xo, scenes, sc, view, np, tile_cull, ray_eval, features):
    cam = xo.make_camera(sc.cameras[view])
    cfg = xo.make_config(dict(scenes.default_render_config(sc), tile_cull=tile_cull))
    arrays = dict(means=sc.means, scales=sc.scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    render, backward = (xo.render_ray, xo.backward_ray) if ray_eval else (xo.render, xo.backward)
    t0 = time.perf_counter()
    r = render(arrays, cam, cfg, np.float32)
    _, dL = scenes.loss_and_grad(sc.loss, r["fwd"]["image"], sc.target(view))
    if features:     # f3: the depth / accumulated-opacity pass and the backward with their (here constant) gradients
        fwd_da, bwd_da = (xo.rasterize_ray_fwd_da, xo.backward_ray_da) if ray_eval else (xo.rasterize_fwd_da, xo.backward_da)
        r["fwd"].update(fwd_da(r["proj"], r["binned"], cam, cfg, np.float32))
        one = np.ones(r["fwd"]["image"].shape[:2], np.float32)
        bwd_da(arrays, r, dL, one, one, cam, cfg, np.float32)
    else:
        backward(arrays, r, dL, cam, cfg, np.float32)
    return time.perf_counter() - t0, r["binned"]["num_pairs"]


def oracle_sample(args):
    """Bounded sample of the bench workload for the CPU legs, sized so that a step is seconds of CPU
    work: the full workload for configs 1-4; for config 5 the same scene at 1/4 linear resolution."""
    from paper_2606_11529_b200 import scenes
    full = scenes.make_scene(args.config)
    W, H = full.cameras[0].width, full.cameras[0].height
    if args.config >= 5:
        w, h = W // 4, H // 4
        sc = scenes.make_scene(args.config, image_override=(w, h))
        desc = f"same scene, all {sc.N} Gaussians, view {args.view}, {w}x{h} image (1/4 linear resolution, same FOV), 1 step"
    else:
        sc, w, h = full, W, H
        desc = f"full workload, {sc.N} Gaussians, {w}x{h}, 1 step"
    return sc, w, h, desc


def run_reference(args):
    """--impl reference: the oracle on the host cores (this tier's reference arm)."""
    if rank_env()[1] != 0:
        return
    import numpy as np
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import xpr_oracle as xo
    from paper_2606_11529_b200 import scenes
    sc, w, h, desc = oracle_sample(args)
    for _ in range(args.warmup):
        oracle_step(xo, scenes, sc, args.view, np, args.tile_cull, args.ray_eval, args.features, args.views)
    t = 0.0
    for _ in range(args.steps):
        dt, I = oracle_step(xo, scenes, sc, args.view, np, args.tile_cull, args.ray_eval, args.features, args.views)
        t += dt
    ms = 1e3 * t / max(args.steps, 1)
    val = (max(1, args.views) * w * h / 1e6) / (ms / 1e3)
    cores = xo.num_threads()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config], "view": args.view, "views": max(1, args.views), "tile_cull": args.tile_cull, "ray_eval": args.ray_eval, "features": args.features, "sample": desc,
                       "pairs": int(I)},
            "gaussians_per_s": sc.N / (ms / 1e3),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# algorithmic work per unit: FP32 lane-ops per pixel-pair
FWD_OPS_VISIT, FWD_OPS_PASS = 8, 9
BWD_OPS_VISIT, BWD_OPS_PASS = 8, 45
# f2 (ray evaluation): d_c 9 + cross 6 + two squared norms 6 + 1 + two thresholds and compares 4
RAY_FWD_OPS_VISIT, RAY_FWD_OPS_PASS = 26, 12
RAY_BWD_OPS_VISIT, RAY_BWD_OPS_PASS = 26, 57
# f3 (depth + accumulated opacity): 2 more lane-ops per blended pair forward, 4 more backward
FEAT_FWD_EXTRA, FEAT_BWD_EXTRA = 2, 4
SMS, LANES_PER_SM = 148, 128


LIN_FWD_OPS_VISIT, LIN_FWD_OPS_PASS = 34, 9   # chord: dx, dy, 4 x (mul, fma, neg), 8 add/sub, 6 min/max, compare, mul; blend: as the Gaussians


def run_linprim(args):
    """f4: the LinPrim step (xpr_lin_project -> xpr_bin_sort_lin -> xpr_lin_rasterize_fwd -> loss gradient ->
    xpr_lin_rasterize_bwd -> xpr_lin_project_bwd), same protocol as the Gaussian step: W warm-up steps, K timed steps
    with the L2 flushed in between, CUDA events per stage, clocks sampled during the timed region."""
    import numpy as np
    import torch
    from paper_2606_11529_b200 import binding as xb, pipeline, scenes
    world, _, local = rank_env()
    if world > 1:
        raise SystemExit("bench.py --linprim: one GPU")
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    xb.lib()
    sc = scenes.make_scene(args.config)
    cam = sc.cameras[args.view]
    if int(cam.model) != 0:
        raise SystemExit("bench.py --linprim: pinhole configs only")
    cfg = dict(scenes.default_render_config(sc), tile_cull=args.tile_cull)
    scales = np.ascontiguousarray(sc.scales * np.float32(args.linprim), np.float32)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    params = (t(sc.means), t(scales), t(sc.quats), t(sc.opacities), t(sc.sh))
    target = t(sc.target(args.view))
    dL = torch.empty_like(target)
    pipe = pipeline.LinPrimPipeline(sc.N, cam, cfg, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    names = ("project", "bin_sort", "rasterize_fwd", "loss_grad", "rasterize_bwd", "project_bwd")

    def rec():
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    def step(events, sync):
        ev = events.append
        ev(rec()); pipe.project(*params)
        ev(rec()); pipe.bin_sort() if sync else pipe.bin_sort_async()
        ev(rec()); pipe.rasterize_fwd()
        ev(rec()); xb.xpr_loss_grad(sc.loss, pipe.image, target, dL)
        ev(rec()); pipe.rasterize_bwd(dL)
        ev(rec()); pipe.project_bwd()
        ev(rec())

    for _ in range(max(args.warmup, 3)):
        step([], True)
    torch.cuda.synchronize()
    n_pairs = pipe.num_pairs
    sampler = ClockSampler(local)
    sampler.start()
    runs = []
    for _ in range(args.steps):
        flush.fill_(1)
        evs = []
        step(evs, False)
        torch.cuda.synchronize()
        runs.append(evs)
    clocks = sampler.stop()
    per_step = np.array([e[0].elapsed_time(e[-1]) for e in runs])
    stage_ms = {n: float(np.mean([e[i].elapsed_time(e[i + 1]) for e in runs])) for i, n in enumerate(names)}
    ms = float(per_step.mean())
    stats = torch.zeros(4, dtype=torch.int64, device=dev)
    xb.xpr_lin_rasterize_stats(pipe.cam, pipe.cfg, pipe.lin_rec, pipe.vals_sorted, pipe.tile_ranges, stats)
    visit, passed, blended, sum_n = [int(v) for v in stats.tolist()]
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    alu_peak = SMS * LANES_PER_SM * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
    ach = (LIN_FWD_OPS_VISIT * visit + LIN_FWD_OPS_PASS * passed) / (stage_ms["rasterize_fwd"] / 1e3) / 1e12
    roofline = {"kernel": "lin_rasterize_fwd_kernel", "bound": "alu", "unit": "T lane-op/s", "peak": alu_peak, "achieved": ach,
                "frac": ach / alu_peak, "traffic": None,
                "algorithmic": "%d x visited + %d x passed lane-ops per (pixel, primitive)" % (LIN_FWD_OPS_VISIT, LIN_FWD_OPS_PASS)}
    mp = cam.width * cam.height / 1e6
    cpu = None
    if not args.no_cpu_baseline:
        sys.path.insert(0, os.path.join(ROOT, "oracle"))
        import xpr_oracle as xo
        arr = dict(means=sc.means, scales=scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
        ocam, ocfg = xo.make_camera(cam), xo.make_config(cfg)
        t0 = time.perf_counter()
        r = xo.render_lin(arr, ocam, ocfg, np.float32)
        _, g = scenes.loss_and_grad(sc.loss, r["fwd"]["image"], sc.target(args.view))
        xo.backward_lin(arr, r, g.astype(np.float32), ocam, ocfg, np.float32)
        dt = time.perf_counter() - t0
        cpu = {"value": mp / dt, "unit": "MP/s", "cores": os.cpu_count(), "kind": "oracle", "seconds": dt,
               "sample": "full workload, %d primitives, %dx%d, 1 step" % (sc.N, cam.width, cam.height)}
    print(json.dumps({
        "metric": "fwd_bwd_megapixels_per_s", "value": mp / (ms / 1e3), "unit": "MP/s", "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config] + " read as octahedra (XPR-LinPrim)", "method": "linprim",
                   "half_axes": "%g x the Gaussian scales" % args.linprim, "view": args.view, "tile_cull": args.tile_cull,
                   "primitives": sc.N, "image": [cam.width, cam.height], "pairs": n_pairs,
                   "l2": "flushed between timed steps (256 MiB write)", "parallelism": "1 GPU"},
        "ms_per_step_stats": {"mean": ms, "median": float(np.median(per_step)), "min": float(per_step.min())},
        "stage_ms": stage_ms, "counts": {"visited": visit, "passed": passed, "blended": blended, "sum_n_contrib": sum_n},
        "roofline": roofline, "clocks": clocks, "e2e": None, "gpu_launches": args.steps * (1 + 11 + 1 + 1 + 1 + 1),
        "cpu_baseline": cpu}))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2606_11529_b200 import binding as xb, pipeline, scenes

    world, rank, local = rank_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --impl ours needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    xb.lib()   # fail loudly if libxpr.so is missing

    sc = scenes.make_scene(args.config)
    cam = sc.cameras[args.view]
    V = max(1, args.views)
    if V > 1 and (args.ray_eval or args.view + V > len(sc.cameras)):
        raise SystemExit("bench.py: --views V needs V cameras in the scene (config 5 has four) and the 2D evaluation")
    cfg = dict(scenes.default_render_config(sc), tile_cull=args.tile_cull, ray_eval=args.ray_eval,
               tile_order=args.tile_order, features=args.features)
    if args.overlap_fill >= 0:
        cfg["overlap_fill"] = args.overlap_fill
    cfg["fuse_loss"] = args.fuse_loss
    params = pipeline.scene_to_device(sc, dev)
    if V > 1:
        target = torch.from_numpy(np.stack([sc.target(args.view + v) for v in range(V)])).to(dev)
        pipe = pipeline.SplatPipeline(sc.N, [sc.cameras[args.view + v] for v in range(V)], cfg, device=dev)
        args.no_plain = True      # the extra plain-path timing is a single-view leg
    else:
        target = torch.from_numpy(sc.target(args.view)).to(dev)
        pipe = pipeline.SplatPipeline(sc.N, cam, cfg, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    dL_buf = torch.empty_like(target)
    if args.features:    # loss + sum gD D + sum gA A with seeded constant gD, gA ~ U[-1, 1] (linear in the features)
        gen = torch.Generator(device="cpu").manual_seed(4000 + args.config)
        vs = (V,) if V > 1 else ()
        pipe.feature_grads = tuple((torch.rand(*vs, cam.height, cam.width, generator=gen) * 2 - 1).to(dev) for _ in range(2))
    feat_grads = pipe.feature_grads or (None, None)

    def loss_grad(image):
        """dL/dimage of the config's loss (sum |I - target| or sum (I - target)^2), one pass (xpr_loss_grad)."""
        xb.xpr_loss_grad(sc.loss, image, target, dL_buf)
        return dL_buf

    fused = pipe.can_fuse_loss()         # loss gradient inside the compositing backward: the loss_grad stage is then empty

    def loss_stage(p):
        return None if fused else loss_grad(p.image)

    def bwd_stage(p, dL):
        if fused:
            p.rasterize_bwd_loss(target, sc.loss)
        else:
            p.rasterize_bwd(dL, *feat_grads)

    stage_names = ("project", "bin_sort", "rasterize_fwd", "loss_grad", "rasterize_bwd", "project_bwd")

    def step(events=None, sync_count=False, stages=True):
        """One fwd+bwd step.  sync_count=True: xpr_bin_sort reads the pair count back (and regrows the pair
        buffers if needed) -- used for the warm-up; the timed steps run fully asynchronously and the count is
        checked against the capacity after the timed region.  stages=False: only the step's first and last event are
        recorded (an event between two stages costs ~2 us of stream time: 13 us per step on config 3)."""
        rec_ev = (lambda: None) if events is None else (lambda: events.append(_rec()))
        ev = rec_ev if stages else (lambda: None)
        rec_ev(); pipe.project(*params)
        if args.ray_eval:                   # pixel_info and the shader record belong to the projection stage
            pipe.pixel_info(); pipe.project_ray()
        ev(); pipe.bin_sort() if sync_count else pipe.bin_sort_async()
        ev(); pipe.rasterize_fwd()
        ev(); dL = loss_stage(pipe)
        ev(); bwd_stage(pipe, dL)
        ev(); pipe.project_bwd()
        rec_ev()

    def _rec():
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step(sync_count=True)
    barrier()
    n_pairs = pipe.num_pairs
    n_cand = pipe.candidates_on_device()
    # our kernels per step: project, emit, passes x onesweep, ranges, rasterize_fwd, rasterize_bwd, project_bwd
    ST = ((pipe.TW + 7) // 8) * ((pipe.TH + 7) // 8)
    tile_passes = max(1, ((max(ST, 1) - 1).bit_length() + 7) // 8)      # 8-bit digits of the supertile id
    # project, bin_sort (compact, 4 depth passes, rank scan, rows, supertile words, tile scan, supertile passes, final),
    # fwd, loss_grad, bwd, project_bwd
    launches_per_step = 1 + (1 + 4 + 1 + 1 + 1 + 1 + tile_passes + 1) + 1 + 1 + 1 + 1
    if fused:
        launches_per_step -= 1              # no loss_grad kernel
    if args.ray_eval:
        launches_per_step += 3              # pixel_info, project_ray, ray_bwd
    if args.features:
        launches_per_step += 1              # depth_bwd
    if pipe.tile_order is not None:
        launches_per_step += 1              # tile_order_kernel at the end of xpr_bin_sort
    n_rows = pipe.rows_on_device()
    n_vis = int(torch.count_nonzero(pipe.tile_count).item())

    sampler = ClockSampler(local)
    sampler.start()
    all_events = []
    barrier()
    timed = []
    for _ in range(args.steps):             # the K timed steps: one event before, one after each step
        flush.fill_(1)                      # L2 flush between timed iterations (outside the event pairs)
        evs = []
        step(evs, stages=False)
        timed.append(evs)
    barrier()
    assert pipe.check_capacity() == n_pairs          # the asynchronous steps produced the same, fitting, pair count
    # a second pass of K steps with an event between the stages: the breakdown.  Every stage is timed ALONE here: the
    # zero-fill of the parameter gradients, which the timed steps above run on a second stream under the forward
    # compositing kernel (pipeline option overlap_fill), is back inside project_bwd, so no stage shares the GPU
    timed_overlap = int(pipe.overlap_fill)
    torch.cuda.synchronize()
    pipe.overlap_fill = 0                   # (every timed step consumed the fill it forked: none is pending)
    for _ in range(args.steps):
        flush.fill_(1)
        evs = []
        step(evs)
        all_events.append(evs)
    barrier()
    pipe.overlap_fill = timed_overlap
    step_ms = [e[0].elapsed_time(e[-1]) for e in timed]
    total_ms = max_over_ranks(float(sum(step_ms)), world, dev)
    ms = total_ms / args.steps
    instrumented_ms = float(np.mean([e[0].elapsed_time(e[-1]) for e in all_events]))
    stage_ms = {n: float(np.mean([e[i].elapsed_time(e[i + 1]) for e in all_events])) for i, n in enumerate(stage_names)}
    stage_ms_median = {n: float(np.median([e[i].elapsed_time(e[i + 1]) for e in all_events])) for i, n in enumerate(stage_names)}
    step_stats = {"mean": float(np.mean(step_ms)), "median": float(np.median(step_ms)), "min": float(np.min(step_ms)),
                  "max": float(np.max(step_ms)), "note": "this rank's K timed steps, one CUDA event before and one after each; ms_per_step is the mean, max over ranks",
                  "instrumented_ms_per_step": instrumented_ms,
                  "stage_ms_note": "stage_ms comes from a second pass of K steps with an event between the stages and every stage alone "
                                   "on the GPU (overlap_fill 0: the 236 B/Gaussian zero-fill inside project_bwd); the events cost stream "
                                   "time and the timed steps run that fill under the forward kernel, so the stages sum to "
                                   "instrumented_ms_per_step, not to ms_per_step"}
    mp = V * cam.width * cam.height / 1e6
    value = aggregate_value(world, mp, ms)

    # roofline of the dominant kernel (largest stage): pixel-pair counts from xpr_rasterize_stats
    stats = torch.zeros(4, dtype=torch.int64, device=dev)
    if args.ray_eval:
        xb.xpr_rasterize_ray_stats(pipe.cam, pipe.cfg, pipe.ray_rec, pipe.conic_opac, pipe.rgb, pipe.lnv,
                                   pipe.pixel_rays, pipe.vals_sorted, pipe.tile_ranges, stats)
    else:
        xb.xpr_rasterize_stats(pipe.cam, pipe.cfg, pipe.shade_rec, pipe.vals_sorted, pipe.tile_ranges, stats)
    fwd_ops = (RAY_FWD_OPS_VISIT, RAY_FWD_OPS_PASS) if args.ray_eval else (FWD_OPS_VISIT, FWD_OPS_PASS)
    bwd_ops = (RAY_BWD_OPS_VISIT, RAY_BWD_OPS_PASS) if args.ray_eval else (BWD_OPS_VISIT, BWD_OPS_PASS)
    kname = "rasterize_ray_%s_kernel" if args.ray_eval else "rasterize_%s_kernel"
    visit, passed, blended, sum_n = [int(v) for v in stats.cpu().tolist()]
    feat_fwd_ops = FEAT_FWD_EXTRA * blended if args.features else 0
    feat_bwd_ops = FEAT_BWD_EXTRA * blended if args.features else 0
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    alu_peak = SMS * LANES_PER_SM * sm_max * 1e6 / 1e12          # T lane-ops/s (FMA = 1 lane-op)
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    sec = lambda n: stage_ms[n] / 1e3
    # 8 B per Gaussian (compact) + 16 B per visible Gaussian per depth pass + 36 B per visible Gaussian
    # (rank scan: index, rectangle, tile count read; two offsets written) + 8 B per row (4 written by rows, 4 read by
    # final) + per supertile word 8 B emitted, 16 B sorted per supertile digit, 8 + 28 B read by final (word; index,
    # depth bits, rectangle, row base of its Gaussian) + 12 B per pair (key + value written once)
    n_words = pipe.words_on_device()
    st_passes = max(1, ((max(1, ((pipe.TW + 7) // 8) * ((pipe.TH + 7) // 8)) - 1).bit_length() + 7) // 8)
    sort_bytes = (8 * sc.N + (4 * 16 + 36) * n_vis + 8 * n_rows + (8 + 16 * st_passes + 36) * n_words + 12 * n_pairs)
    rooflines = {
        "rasterize_fwd": {"kernel": (kname % "fwd") + ("<FEAT>" if args.features else ""), "bound": "alu",
                          "unit": "T lane-op/s", "peak": alu_peak,
                          "achieved": (fwd_ops[0] * visit + fwd_ops[1] * passed + feat_fwd_ops) / sec("rasterize_fwd") / 1e12},
        "rasterize_bwd": {"kernel": (kname % "bwd") + ("<FEAT>" if args.features else ""), "bound": "alu",
                          "unit": "T lane-op/s", "peak": alu_peak,
                          "achieved": (bwd_ops[0] * sum_n + bwd_ops[1] * blended + feat_bwd_ops) / sec("rasterize_bwd") / 1e12},
        "bin_sort": {"kernel": "xpr_bin_sort%s (compact, 4 depth passes on Gaussians, rank scan, rows, supertile words, "
                               "tile scan, %d supertile pass(es) on words, final)" % ("_cull" if args.tile_cull else "", tile_passes), "bound": "hbm", "unit": "GB/s", "peak": hbm_peak,
                     "achieved": sort_bytes / sec("bin_sort") / 1e9, "algorithmic_bytes": sort_bytes},
    }
    traffic = {}
    try:   # dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed ncu captures (profiles/ncu_traffic.md)
        key = "config%d%s" % (args.config, "_ray" if args.ray_eval else "_feat" if args.features else "")
        for ln in open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")).read().splitlines()[1:]:
            w, stage, b = ln.split(",")
            if w == key:
                traffic[stage] = int(b)
    except Exception:
        pass
    for name, r in rooflines.items():
        r["frac"] = r["achieved"] / r["peak"]
        if r["bound"] == "hbm":
            r["frac_of_nominal_8TBs"] = r["achieved"] / 8000.0
        r["traffic"] = traffic.get(name)
        r["traffic_source"] = ("profiles/ncu_traffic.csv (dram__bytes_read.sum + dram__bytes_write.sum of a committed ncu --set full "
                               "capture of this workload, see profiles/ncu_traffic.md; not measured by this run)"
                               if traffic.get(name) is not None else None)
        r["peak_source"] = "MEASURED_PEAKS.json" if peaks else "fallback (B200_PROFILING.md)"
        r["ms_per_launch"] = stage_ms[name]
    dom = max(rooflines, key=lambda n: stage_ms[n])
    roof = rooflines[dom]

    # the plain north_star path (rectangle-overlap binning, no tile_cull) on the same workload, same protocol, when the
    # headline run used tile_cull: its own pipeline and buffers, K timed steps with the L2 flushed in between
    plain_path = None
    if args.tile_cull and not args.no_plain:
        cfg0 = dict(cfg, tile_cull=0)
        pipe0 = pipeline.SplatPipeline(sc.N, cam, cfg0, device=dev)
        pipe0.feature_grads = pipe.feature_grads

        def step0(sync):
            pipe0.project(*params)
            if args.ray_eval:
                pipe0.pixel_info(); pipe0.project_ray()
            pipe0.bin_sort() if sync else pipe0.bin_sort_async()
            pipe0.rasterize_fwd()
            bwd_stage(pipe0, loss_stage(pipe0))
            pipe0.project_bwd()
        for _ in range(3):
            step0(True)
        barrier()
        t0 = []
        for _ in range(args.steps):
            flush.fill_(1)
            a = _rec(); step0(False); b = _rec()
            torch.cuda.synchronize()
            t0.append(a.elapsed_time(b))
        n0 = pipe0.check_capacity()
        ms0 = max_over_ranks(float(np.mean(t0)), world, dev)
        plain_path = {"tile_cull": 0, "pairs": n0, "ms_per_step": ms0, "ms_per_step_median": float(np.median(t0)),
                      "ms_per_step_min": float(np.min(t0)), "value": aggregate_value(world, mp, ms0), "unit": UNIT}
        del pipe0

    # the same step captured once in a CUDA graph and replayed (no host work between the 15 launches)
    graph_ms = None
    if not args.no_graph:
        try:
            g = pipe.capture_step(*params, target, sc.loss, pixel_info=bool(args.ray_eval))
            for _ in range(3):
                g.replay()
            barrier()
            t_ms = 0.0
            for _ in range(args.steps):
                flush.fill_(1)
                a = _rec(); g.replay(); b = _rec()
                torch.cuda.synchronize()
                t_ms += a.elapsed_time(b)
            assert pipe.check_capacity() == n_pairs
            graph_ms = max_over_ranks(t_ms, world, dev) / args.steps
        except Exception as e:      # capture unsupported in this environment: report, do not hide
            graph_ms = "unavailable: %s" % (str(e).splitlines()[0][:120],)

    featn = None
    if args.featn > 0 and not args.ray_eval:     # N-channel features: the two kernels alone, warm L2
        gen = torch.Generator(device="cpu").manual_seed(5000 + args.featn)
        feat = torch.randn(sc.N, args.featn, generator=gen).to(dev)
        gF = (torch.rand(cam.height, cam.width, args.featn, generator=gen) * 2 - 1).to(dev)
        F_img, g_feat = torch.empty_like(gF), torch.empty_like(feat)

        def _time(fn, n=20):
            for _ in range(3):
                fn()
            a = _rec()
            for _ in range(n):
                fn()
            b = _rec()
            torch.cuda.synchronize()
            return a.elapsed_time(b) / n
        featn = {"C": args.featn,
                 "fwd_ms": _time(lambda: pipe.rasterize_featn_fwd(feat, F_img)),
                 "bwd_ms": _time(lambda: pipe.rasterize_featn_bwd(feat, gF, g_feat)),
                 "how": "20 back-to-back launches each, CUDA events, warm L2, after the timed steps"}

    cub_compare = None
    if args.sort_compare:
        import ctypes as C
        from paper_2606_11529_b200 import build as xbuild
        cl = C.CDLL(xbuild.build_cub_compare())
        cl.xpr_cubcmp_sort_pairs.restype = C.c_int32
        I = n_pairs
        ks, vs = pipe.keys_sorted[:I].clone(), pipe.vals_sorted[:I].clone()
        # the pairs in EMISSION order (Gaussian by Gaussian, row-major inside its rectangle = ascending tile id):
        # a stable sort of the sorted pairs by Gaussian index restores it
        order = torch.argsort(vs.to(torch.int64), stable=True)
        kin, vin = ks[order].contiguous(), vs[order].contiguous()
        kout, vout = torch.empty_like(kin), torch.empty_like(vin)
        end_bit = 32 + max(1, (pipe.T - 1).bit_length())
        nbytes = C.c_size_t(0)
        stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
        p = lambda t: C.c_void_p(t.data_ptr())
        assert cl.xpr_cubcmp_sort_pairs(C.c_int64(I), p(kin), p(vin), p(kout), p(vout), None, C.byref(nbytes), 0, end_bit, stream) == 0
        temp = torch.empty(max(int(nbytes.value), 1), dtype=torch.uint8, device=dev)
        run = lambda: cl.xpr_cubcmp_sort_pairs(C.c_int64(I), p(kin), p(vin), p(kout), p(vout), p(temp), C.byref(nbytes), 0, end_bit, stream)
        for _ in range(3):
            assert run() == 0
        torch.cuda.synchronize()
        same = bool(torch.equal(kout, ks) and torch.equal(vout, vs))     # both are THE stable sort by key
        ts = []
        for _ in range(max(args.steps, 5)):
            flush.fill_(1)
            a = _rec(); run(); b = _rec()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        ts.sort()
        cub_compare = {"pairs": I, "key_bits_sorted": end_bit, "cub_sort_pairs_ms": {"median": ts[len(ts) // 2], "min": ts[0]},
                       "cub_temp_bytes": int(nbytes.value), "output_equals_xpr_bin_sort": same,
                       "xpr_bin_sort_ms": stage_ms["bin_sort"],
                       "note": "CUB sorts (u64 key, u32 value) pairs that already exist in memory; xpr_bin_sort starts from the "
                               "projection outputs: it also compacts, scans, culls, generates the pairs and writes tile_ranges"}
        del ks, vs, kin, vin, kout, vout, temp, order

    clocks = sampler.stop()      # sampled (every 20 ms) over the timed steps and the graph replays

    # end to end through the public API with HOST buffers: H2D of the parameters, the step, D2H of results
    e2e = None
    if not args.no_e2e:
        host_in = [torch.from_numpy(a).pin_memory() for a in (sc.means, sc.scales, sc.quats, sc.opacities, sc.sh)]
        dev_in = [torch.empty_like(p) for p in params]
        outs = [pipe.image, pipe.g_means, pipe.g_scales, pipe.g_quats, pipe.g_opacities, pipe.g_sh]
        if args.features:
            outs += [pipe.depth_img, pipe.alpha_img]
        host_out = [torch.empty(o.shape, dtype=o.dtype).pin_memory() for o in outs]
        h2d = sum(t.numel() * t.element_size() for t in host_in)
        d2h = sum(t.numel() * t.element_size() for t in host_out)

        def run_step(inputs):
            pipe.project(*inputs)
            if args.ray_eval:
                pipe.pixel_info(); pipe.project_ray()
            pipe.bin_sort_async(); pipe.rasterize_fwd()
            bwd_stage(pipe, loss_stage(pipe)); pipe.project_bwd()

        def e2e_step():       # one stream: copy in, step, copy out (the latency of a single step)
            for d, h in zip(dev_in, host_in):
                d.copy_(h, non_blocking=True)
            run_step(dev_in)
            for h, o in zip(host_out, outs):
                h.copy_(o, non_blocking=True)

        for _ in range(2):
            e2e_step()
        barrier()
        k = max(3, args.steps)
        t_ms = 0.0
        for _ in range(k):
            flush.fill_(1)
            a = _rec(); e2e_step(); b = _rec()
            torch.cuda.synchronize()
            t_ms += a.elapsed_time(b)
        lat_ms = max_over_ranks(t_ms, world, dev) / k

        # the same K steps as a three-stage software pipeline: the H2D copy of step i+1 and the D2H copy of step i-1
        # run on their own streams (PCIe is full duplex) under the kernels of step i.  Inputs and the outputs'
        # staging copies are double-buffered; every step still copies all its inputs in and all its results out.
        s_c = torch.cuda.current_stream()
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        dev_in2 = [dev_in, [torch.empty_like(p) for p in params]]
        stage = [[torch.empty_like(o) for o in outs] for _ in range(2)]

        def pipelined(n):
            ev_in, ev_c, ev_out = [None] * n, [None] * n, [None] * n
            start = torch.cuda.Event(enable_timing=True); start.record(s_c)
            s_in.wait_event(start); s_out.wait_event(start)
            for i in range(n):
                bsel = i % 2
                with torch.cuda.stream(s_in):
                    if i >= 2:
                        s_in.wait_event(ev_c[i - 2])            # the kernels that read this input buffer are done
                    for d, h in zip(dev_in2[bsel], host_in):
                        d.copy_(h, non_blocking=True)
                    ev_in[i] = torch.cuda.Event(); ev_in[i].record(s_in)
                s_c.wait_event(ev_in[i])
                run_step(dev_in2[bsel])
                if i >= 2:
                    s_c.wait_event(ev_out[i - 2])               # this staging buffer has left for the host
                for st_, o in zip(stage[bsel], outs):
                    st_.copy_(o, non_blocking=True)
                ev_c[i] = torch.cuda.Event(); ev_c[i].record(s_c)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_c[i])
                    for h, st_ in zip(host_out, stage[bsel]):
                        h.copy_(st_, non_blocking=True)
                    ev_out[i] = torch.cuda.Event(); ev_out[i].record(s_out)
            end = torch.cuda.Event(enable_timing=True)
            s_c.wait_stream(s_out); s_c.wait_stream(s_in)
            end.record(s_c)
            torch.cuda.synchronize()
            return start.elapsed_time(end)

        pipelined(3)
        barrier()
        t_ms = max_over_ranks(pipelined(k), world, dev)
        assert pipe.check_capacity() == n_pairs
        pipe_ms = t_ms / k
        best = min(pipe_ms, lat_ms)      # tiny configs: the events of the pipeline cost more than the overlap saves
        e2e = {"value": aggregate_value(world, mp, best), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": best, "steps": k,
               "how": ("K steps as a 3-stage pipeline (H2D | kernels | D2H on three streams, double-buffered)"
                       if pipe_ms <= lat_ms else "K steps on one stream (copy in, kernels, copy out)")
                      + "; every step copies all inputs from and all results (image + parameter gradients) to pinned "
                        "host memory",
               "pipelined_ms_per_step": pipe_ms, "single_stream_ms_per_step": lat_ms}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        sys.path.insert(0, os.path.join(ROOT, "oracle"))
        import xpr_oracle as xo
        osc, w, h, desc = oracle_sample(args)
        dt, _ = oracle_step(xo, scenes, osc, args.view, np, args.tile_cull, args.ray_eval, args.features, args.views)
        cpu = {"value": (V * w * h / 1e6) / dt, "unit": UNIT, "cores": xo.num_threads(), "kind": "oracle", "sample": desc,
               "seconds": dt}
        if args.config <= 2:     # also one thread for the two small configs (a fresh process: OMP_NUM_THREADS=1)
            code = ("import sys, time, numpy as np; sys.path[:0] = [%r, %r]; import bench, xpr_oracle as xo; "
                    "from paper_2606_11529_b200 import scenes; sc = scenes.make_scene(%d); "
                    "dt, _ = bench.oracle_step(xo, scenes, sc, %d, np, %d, %d, %d); print(dt, xo.num_threads())"
                    % (ROOT, os.path.join(ROOT, "oracle"), args.config, args.view, args.tile_cull, args.ray_eval, args.features))
            try:
                out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600,
                                     env=dict(os.environ, OMP_NUM_THREADS="1"))
                dt1, th1 = out.stdout.split()[-2:]
                cpu["one_thread"] = {"value": (w * h / 1e6) / float(dt1), "unit": UNIT, "cores": int(th1), "seconds": float(dt1)}
            except Exception as e:
                cpu["one_thread"] = "unavailable: %s" % (str(e)[:100],)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": WORKLOADS[args.config], "view": args.view, "gaussians": sc.N,
                           "image": [cam.width, cam.height], "views": V, "tile_cull": args.tile_cull, "ray_eval": args.ray_eval, "features": args.features, "tile_order": int(pipe.tile_order is not None), "fuse_loss": int(fused), "overlap_fill": int(pipe.overlap_fill), "pairs": n_pairs,
                           "candidate_pairs": n_cand, "rows": n_rows, "supertile_words": n_words, "visible_gaussians": n_vis,
                           "sort_passes": {"depth_digits_on_gaussians": 4, "supertile_digits_on_words": tile_passes,
                                           "on_pairs": 0},
                           "l2": "flushed between timed steps (256 MiB write); inputs (236 MB) also exceed L2",
                           "parallelism": "replicas only" if world > 1 else "1 GPU"},
                "gaussians_per_s": world * V * sc.N / (ms / 1e3), "ms_per_step_stats": step_stats, "stage_ms": stage_ms,
                "stage_ms_median": stage_ms_median, "plain_path": plain_path,
                "pixel_pairs": {"visited": visit, "passed_gate": passed, "blended": blended, "sum_n_contrib": sum_n},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
                "cuda_graph_ms_per_step": graph_ms, "featn": featn, "cub_compare": cub_compare, "roofline": roof, "rooflines": rooflines, "cpu_baseline": cpu}
        print(json.dumps(line), flush=True)
        if args.stages:
            print(json.dumps(stage_ms, indent=1), file=sys.stderr)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    elif a.linprim > 0:
        run_linprim(a)
    else:
        run_ours(a)
