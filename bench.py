#!/usr/bin/env python
"""bench.py - forward+backward Mrays/s of the sparse-voxel tile rasterizer on config C4 (BASELINE.json
configs[3], the Mip-NeRF-360-shaped 4M-voxel scene the metric is quoted on), one process per GPU.

A "step" is one training view through the whole hot path: svr_preprocess (project, key build, sort, ranges,
per-view colours) -> svr_forward -> svr_loss_grad -> svr_backward (+ SH backward, w_max), cameras taken
round-robin from the config's 8 views. Inputs are seeded synthetic (svr_inputs), resident in HBM for `value`;
`e2e` goes through svr_train_view_host with the step's inputs (camera + target image) in pinned HOST memory and
the loss read back to the host inside the timed region. The scene parameters (928 MB) and the sorted lists
are far larger than the 126 MB L2, so no explicit L2 flush is needed between iterations.

--impl reference times the CPU oracle (oracle/, fp64, OpenMP) on a bounded sample of the same workload.
N > 1 (torchrun): independent replicas (the path has no exchange step: DESIGN.md "Multi-GPU"), weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# algorithmic work per ray-voxel hit: forward 125 flop, backward 250 flop
FLOP_PER_FWD_HIT = 125.0
FLOP_PER_BWD_HIT = 250.0
FP32_LANES_PER_SM = 128


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return d, "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


def git_blob_hash(path: str) -> str:
    """`git hash-object` of a file (sha1 over "blob <len>\\0" + content), computed here so that no git checkout is needed."""
    import hashlib
    with open(path, "rb") as f:
        data = f.read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def ncu_counters(kernel: str):
    """Counters of one launch of a compositing kernel on full-size C4 from the committed ncu capture (profiles/r3_counters.csv,
    see r3_counters.md): DRAM bytes, L2 reduction sectors, executed FFMA / FADD / FMUL thread instructions per elapsed cycle.
    They are NOT measured by this run; `stale` says whether composite.cu changed since the capture (git blob hash)."""
    path = os.path.join(ROOT, "profiles", "r3_counters.csv")
    if not os.path.exists(path):
        return None
    with open(path) as fh:
        lines = [ln.strip() for ln in fh if ln.strip() and not ln.startswith("#")]
    cols = lines[0].split(",")
    for ln in lines[1:]:
        row = dict(zip(cols, ln.split(",")))
        if row["kernel"] == kernel:
            now = git_blob_hash(os.path.join(ROOT, "paper_2511_02510_b200", "csrc", "composite.cu"))
            row["stale"] = now != row["composite_cu_blob"]
            return row
    return None


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index: int):
        self.idx = device_index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.idx)], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                smax.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample_run(cfg, cam, n_rays: int, seed: int):
    """The CPU oracle as it stands (bucketed mode, fp64, OpenMP) on n_rays seeded rays: forward + backward."""
    import oracle
    rng = np.random.default_rng(seed)
    xy = np.stack([rng.integers(0, cam.W, n_rays), rng.integers(0, cam.H, n_rays)], axis=1).astype(np.int32)
    G = rng.normal(0, 1.0 / (3 * cam.W * cam.H), size=(n_rays, 3))
    t0 = time.perf_counter()
    oracle.render(cfg.scene, cam, cfg.K, mode="bucketed", xy=xy)
    oracle.backward(cfg.scene, cam, cfg.K, G, mode="bucketed", xy=xy)
    return time.perf_counter() - t0


def run_reference(args):
    """--impl reference: the oracle on this box's host cores, same metric/config; each step is a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from svr_inputs import make_config
    oracle.build()
    cfg = make_config(args.workload, n_voxels=args.n_voxels, res_scale=args.res_scale)
    # the oracle does ~23 k rays/s on 16 cores: 2.5 M rays in all keep K steps within about two minutes
    n_rays = args.ref_rays if args.ref_rays else max(5_000, min(100_000, 2_500_000 // max(args.steps, 1)))
    for i in range(args.warmup if args.warmup < 2 else 1):
        oracle_sample_run(cfg, cfg.cameras[i % len(cfg.cameras)], min(n_rays, 2000), 900 + i)
    total = 0.0
    for i in range(args.steps):
        total += oracle_sample_run(cfg, cfg.cameras[i % len(cfg.cameras)], n_rays, 1000 + i)
    value = n_rays * args.steps / total / 1e6
    cores = oracle.num_threads()
    sample = f"{n_rays} seeded rays per step (of {cfg.cameras[0].W * cfg.cameras[0].H} per view), bucketed fp64 oracle, forward+backward"
    line = {"impl": "reference", "metric": "fwd+bwd Mrays/s", "value": value, "unit": "Mrays/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args),
            "cpu_baseline": {"value": value, "unit": "Mrays/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "Mrays/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def camera_index(step: int, rank: int, n_cams: int) -> int:
    """Replica `rank` walks the config's cameras round-robin starting at camera `rank` (no data-path exchange)."""
    return (step + rank) % n_cams


def max_over_ranks(ms: float, world: int, device) -> float:
    """Device-timed milliseconds -> max over ranks (the whole job is as slow as its slowest replica)."""
    if world <= 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(rays_per_step: int, steps: int, world: int, ms: float) -> float:
    """Whole-job Mrays/s: every rank processed `steps` views in the max-over-ranks time."""
    return rays_per_step * steps * world / (ms * 1e-3) / 1e6


def morton_order(sc):
    """Permutation that sorts the voxels by the Morton code of their cell at the finest level (z-order of the octree)."""
    ij = sc.ijkl.astype(np.uint64)
    shift = (np.uint64(sc.max_level) - ij[:, 3]).astype(np.uint64)
    code = np.zeros(sc.n, dtype=np.uint64)
    for b in range(sc.max_level):
        for a in range(3):
            code |= (((ij[:, a] << shift) >> np.uint64(b)) & np.uint64(1)) << np.uint64(3 * b + a)
    return np.argsort(code, kind="stable")


def workload_config(cfg, args):
    cam = cfg.cameras[0]
    name = cfg.name + (" (voxels stored in Morton order: NOT the metric's config)" if args.scene_order == "morton" else "")
    return {"workload": f"{name}: {cfg.scene.n} voxels, {cam.W}x{cam.H}, {len(cfg.cameras)} cameras round-robin, K={cfg.K}, "
                        f"SH degree {cfg.scene.sh_degree}, T_min={cfg.T_min}, gamma={cfg.gamma}, backward emits w_max and writes the gradients (grad_overwrite)",
            "seed": cfg.seed, "rays_per_step": cam.W * cam.H,
            "l2": "inputs larger than L2 (scene parameters 928 MB at full size); no explicit flush",
            "parallelism": f"replicas x{args.gpus} (no data-path collective)"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=64)
    ap.add_argument("--warmup", type=int, default=4)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4")
    ap.add_argument("--n-voxels", type=int, default=None, help="reduced copy of the workload (debugging only)")
    ap.add_argument("--res-scale", type=float, default=1.0)
    ap.add_argument("--ref-rays", type=int, default=None,
                    help="rays per step of the CPU oracle sample (default: sized so that the whole run takes about two minutes)")
    ap.add_argument("--cpu-baseline-rays", type=int, default=100_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--scene-order", default="config", choices=["config", "morton"],
                    help="config: the storage order the workload recipe gives (random: BASELINE's configs); morton: the same voxels "
                         "stored in octree (Morton) order, as a trainer that keeps its octree sorted would pass them (context only)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2511_02510_b200 as pkg          # raises if libsvr.so is missing: no fallback
    from svr_inputs import make_config

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

    cfg = make_config(args.workload, n_voxels=args.n_voxels, res_scale=args.res_scale)
    sc, cams = cfg.scene, cfg.cameras
    if args.scene_order == "morton":
        order = morton_order(sc)
        sc.ijkl, sc.raw, sc.sh = sc.ijkl[order], sc.raw[order], sc.sh[order]
    W, H = cams[0].W, cams[0].H
    rays = W * H
    ctx = pkg.Context(local_rank, workspace_budget_bytes=cfg.workspace_budget_bytes)
    stream = ctx.stream
    vox = pkg.Voxels.from_scene(sc, device=dev)
    ccams = [pkg.make_camera(c) for c in cams]
    g_raw = torch.zeros((sc.n, 8), dtype=torch.float32, device=dev)
    g_sh = torch.zeros((sc.n, sc.n_basis, 3), dtype=torch.float32, device=dev)
    w_max = torch.zeros(sc.n, dtype=torch.float32, device=dev)
    image = torch.empty((H, W, 3), dtype=torch.float32, device=dev)
    depth = torch.empty((H, W), dtype=torch.float32, device=dev)
    Tf = torch.empty((H, W), dtype=torch.float32, device=dev)
    dL = torch.empty((H, W, 3), dtype=torch.float32, device=dev)
    loss = torch.empty(1, dtype=torch.float32, device=dev)

    # targets: seeded noise-perturbed renders (config recipe), one per camera, device + pinned host copies
    targets, targets_host = [], []
    for i, c in enumerate(ccams):
        fr = ctx.svr_preprocess(vox, c)
        ctx.svr_forward(fr, cfg.K, cfg.T_min, image=image, want_aux=False, record=False)
        ctx.synchronize()
        fr.release()
        rng = np.random.Generator(np.random.PCG64(cfg.seed * 100 + i))
        noise = torch.from_numpy(rng.normal(0, cfg.target_noise, size=(H, W, 3)).astype(np.float32))
        t_host = torch.clamp(image.cpu() + noise, 0.0, 1.0).contiguous().pin_memory()
        targets_host.append(t_host)
        targets.append(t_host.to(dev))

    def step(i):
        k = camera_index(i, rank, len(ccams))
        ctx.svr_loss_prepare(targets[k])        # target-only part of the loss: second stream, beside preprocess + forward
        fr = ctx.svr_preprocess(vox, ccams[k])
        ctx.svr_forward(fr, cfg.K, cfg.T_min, image=image, depth=depth, T_final=Tf)
        ctx.svr_loss_grad(image, targets[k], cfg.gamma, dL=dL, loss=loss)
        ctx.svr_backward(fr, cfg.K, dL, image, g_raw, g_sh, cfg.T_min, w_max=w_max if cfg.emit_wmax_in_backward else None,
                         overwrite=True)     # one view per step: gradients written, not summed (no zero fill between steps)
        fr.release()

    def step_accumulate(i):
        """The ABI's default gradient mode: svr_backward ADDS into grad_raw / grad_sh, so a one-view step zero-fills both first."""
        k = camera_index(i, rank, len(ccams))
        ctx.svr_loss_prepare(targets[k])
        fr = ctx.svr_preprocess(vox, ccams[k])
        ctx.svr_forward(fr, cfg.K, cfg.T_min, image=image, depth=depth, T_final=Tf)
        ctx.svr_loss_grad(image, targets[k], cfg.gamma, dL=dL, loss=loss)
        g_raw.zero_()
        g_sh.zero_()
        ctx.svr_backward(fr, cfg.K, dL, image, g_raw, g_sh, cfg.T_min, w_max=w_max if cfg.emit_wmax_in_backward else None,
                         overwrite=False)
        fr.release()

    def render_step(i):
        k = camera_index(i, rank, len(ccams))
        fr = ctx.svr_preprocess(vox, ccams[k])
        ctx.svr_forward(fr, cfg.K, cfg.T_min, image=image, want_aux=False, record=False)      # render only: no backward follows
        fr.release()

    def e2e_step(i):
        k = camera_index(i, rank, len(ccams))
        return ctx.svr_train_view_host(vox, ccams[k], cfg.K, cfg.gamma, targets_host[k], g_raw, g_sh,
                                       w_max=w_max if cfg.emit_wmax_in_backward else None, T_min=cfg.T_min, overwrite=True)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, sampler=None):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        if sampler:
            sampler.start()
        with torch.cuda.stream(stream):
            e0.record(stream)
            for i in range(steps):
                fn(i)
            e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        clocks = sampler.stop() if sampler else None
        return max_over_ranks(ms, world, dev), clocks

    # set-up, not warm-up: one untimed pass over the cameras so that every camera's workspace blocks exist in the library's
    # cache (a camera's first recording pass allocates its record buffers from the driver; sizes repeat afterwards)
    for i in range(len(ccams)):
        step(i)
    for i in range(args.warmup):
        step(i)
    torch.cuda.synchronize()
    torch.cuda.reset_peak_memory_stats(dev)

    # ---- timed region: K steps of the whole path (no stage timers: `value` carries no event-record overhead) ----
    launches0 = ctx.kernel_launches
    ms_total, clocks = timed(step, args.steps, ClockSampler(local_rank))
    launches = ctx.kernel_launches - launches0
    value = aggregate_value(rays, args.steps, world, ms_total)
    # ---- the same K steps again with stage timers (CUDA events on the library's stream around every stage) ----
    ctx.svr_get_stage_times(reset=True)
    ctx.svr_set_stage_timing(True)
    ms_staged, _ = timed(step, args.steps)
    stage = ctx.svr_get_stage_times(reset=True)
    ctx.svr_set_stage_timing(False)

    # ---- the same steps in the ABI's default accumulate mode, zero fill of both gradient arrays included ----
    with torch.cuda.stream(stream):         # torch's zero fills go on the library's stream
        for i in range(3):
            step_accumulate(i)
    ms_acc, _ = timed(step_accumulate, args.steps)
    value_accumulate = aggregate_value(rays, args.steps, world, ms_acc)

    # ---- one pass over the cameras with w_max cleared first (the first views after a prune / subdivide step pay the
    # atomicMax of every voxel's first sighting; in steady state most hits only read) ----
    w_max.zero_()
    ms_cold, _ = timed(step, len(ccams))
    ms_cold /= len(ccams)

    # ---- render-only FPS (preprocess + forward, w_max off) ----
    for i in range(3):
        render_step(i)
    ms_render, _ = timed(render_step, args.steps)
    render_fps = args.steps * world / (ms_render * 1e-3)

    # ---- end to end through the host-buffer entry point ----
    for i in range(3):
        e2e_step(i)
    ms_e2e, _ = timed(e2e_step, args.steps)
    e2e_value = aggregate_value(rays, args.steps, world, ms_e2e)

    peak_vram = int(torch.cuda.max_memory_allocated(dev)) + int(ctx.workspace_peak_bytes)

    # ---- context (not part of `value`): a whole training iteration = the step + the fused Adam update of both parameter
    # tensors, which also clears the gradients the next backward accumulates into. lr = 0: the parameters do not move. ----
    adam_state = [torch.zeros_like(t.view(-1)) for t in (vox.raw, vox.raw, vox.sh, vox.sh)]
    it_no = [0]

    def train_iter(i):
        step(i)
        it_no[0] += 1
        ctx.svr_adam_step(vox.raw.view(-1), g_raw.view(-1), adam_state[0], adam_state[1], 0.0, 0.9, 0.999, 1e-8, it_no[0], zero_grad=True)
        ctx.svr_adam_step(vox.sh.view(-1), g_sh.view(-1), adam_state[2], adam_state[3], 0.0, 0.9, 0.999, 1e-8, it_no[0], zero_grad=True)

    for i in range(3):
        train_iter(i)
    ms_iter, _ = timed(train_iter, args.steps)
    del adam_state

    # ---- work counters (outside the timed region): hits / tests per view ----
    stats = []
    for k in sorted({camera_index(i, rank, len(ccams)) for i in range(args.steps)}):
        fr = ctx.svr_preprocess(vox, ccams[k])
        st = ctx.svr_forward_stats(fr, cfg.K, cfg.T_min)
        st["entries"] = fr.n_entries
        fr.release()
        stats.append(st)
    hits = float(np.mean([s["hits"] for s in stats]))
    tests = float(np.mean([s["slab_tests"] for s in stats]))
    staged = float(np.mean([s["entries_staged"] for s in stats]))

    peaks, peak_src = measured_peaks()
    micro = ctx.svr_measure_peaks()        # FP32 FFMA / FFMA2 TFLOP/s, L2 red.v4 G/s, warp-instruction issue G/s (outside the timed regions)
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    fp32_peak = n_sm * FP32_LANES_PER_SM * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12    # TFLOP/s
    stage_ms = {k: v[0] / args.steps for k, v in stage.items() if v[1] > 0}       # per step (a stage may launch twice)
    dom = max(stage_ms, key=stage_ms.get)
    flop = {"forward_composite": FLOP_PER_FWD_HIT, "backward_composite": FLOP_PER_BWD_HIT}
    full_c4 = args.workload == "C4" and args.n_voxels is None and args.res_scale == 1.0

    def alu_roofline(kernel):
        """FP32 roofline entry of a compositing kernel: algorithmic flops per launch / live stage time, against the FP32 peak;
        the counters of the committed ncu capture (DRAM traffic, executed-FP32 fraction) next to it when this is full-size C4."""
        achieved = hits * flop[kernel] / (stage_ms[kernel] * 1e-3) / 1e12
        c = ncu_counters(kernel) if full_c4 else None
        traffic = float(c["dram_bytes_per_launch"]) if c else None
        red_sectors = float(c["l2_red_sectors_per_launch"]) if c else None
        # SURVEY 8(d) fraction (i): executed FP32 thread instructions per elapsed cycle, (2 ffma + fadd + fmul) / (SMs x 128 lanes x 2)
        frac_exec = ((2.0 * float(c["ffma_per_cycle"]) + float(c["fadd_per_cycle"]) + float(c["fmul_per_cycle"])) / (n_sm * FP32_LANES_PER_SM * 2)) if c else None
        return {"kernel": kernel, "bound": "alu", "achieved": achieved, "peak": fp32_peak, "unit": "TFLOP/s",
                "frac": achieved / fp32_peak, "traffic": traffic,
                "frac_executed_fp32": frac_exec,
                "traffic_source": (f"profiles/r3_counters.csv (ncu --set full capture, not this run; composite.cu blob {c['composite_cu_blob'][:12]}, "
                                   f"{'STALE: composite.cu changed since' if c['stale'] else 'matches this build'})") if c else None,
                "peak_source": f"{n_sm} SMs x 128 FP32 lanes x 2 x sm_max_mhz, clocks {peak_src}",
                "peak_measured": micro["fp32_ffma_tflops"], "peak_measured_ffma2": micro["fp32_ffma2_tflops"],
                "frac_of_measured_peak": achieved / micro["fp32_ffma_tflops"],
                "issue_peak_measured_gwarp_inst_per_s": micro["issue_gwarp_inst_per_s"],
                "l2_red_v4_peak_measured_g_per_s": micro["l2_red_v4_gops"],
                "l2_red_sectors_per_launch": red_sectors,
                "l2_red_rate_g_per_s": (red_sectors / (stage_ms[kernel] * 1e-3) / 1e9) if red_sectors else None,
                "algorithmic": f"{hits:.4g} ray-voxel hits/view x {flop[kernel]:.0f} flop",
                "kernel_ms": stage_ms[kernel], "slab_tests_per_hit": tests / max(hits, 1.0)}

    if dom in flop:
        roofline = alu_roofline(dom)
    else:   # an HBM-bound stage dominates (not expected): report bytes moved by the sort
        bytes_ = staged * 170.0
        achieved = bytes_ / (stage_ms[dom] * 1e-3) / 1e9
        roofline = {"kernel": dom, "bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": achieved / peaks["hbm_gbs"], "traffic": None, "kernel_ms": stage_ms[dom]}
    roofline_forward = alu_roofline("forward_composite") if "forward_composite" in stage_ms else None
    # the driver's record keeps `roofline` whole: the half of the metric that is not `value` rides in it too
    roofline["render_fps"] = render_fps
    roofline["peak_vram_bytes"] = peak_vram
    roofline["step_flop_frac"] = (hits * (FLOP_PER_FWD_HIT + FLOP_PER_BWD_HIT) / (ms_total / args.steps * 1e-3) / 1e12) / fp32_peak

    line = {"metric": "fwd+bwd Mrays/s", "value": value, "unit": "Mrays/s", "render_fps": render_fps, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": workload_config(cfg, args),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "Mrays/s", "ms_per_step": ms_e2e / args.steps,
                    "h2d_bytes_per_step": int(targets_host[0].numel() * 4 + 92), "d2h_bytes_per_step": 4,
                    "note": "svr_train_view_host: camera + target image from pinned host memory, the 4-byte loss read back; the gradients and "
                            "w_max stay on the device by design (they feed the device-side svr_adam_step / svr_prune_step)"},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "roofline_forward": roofline_forward,
            "value_accumulate": {"value": value_accumulate, "unit": "Mrays/s", "ms_per_step": ms_acc / args.steps,
                                 "what": "the same step with grad_overwrite = 0 (the ABI's default: gradients accumulate) and the zero "
                                         "fill of grad_raw / grad_sh it needs before a one-view step"},
            "ms_per_step_with_stage_timers": ms_staged / args.steps,
            "cold_w_max": {"ms_per_step": ms_cold, "what": "one pass over the cameras right after w_max was cleared (every voxel's first sighting "
                                                           "takes the atomicMax path); `value` is the steady state between two adaptation steps"},
            "work_per_view": {"hits": hits, "slab_tests": tests, "entries_staged": staged,
                              "list_entries": float(np.mean([s["entries"] for s in stats])),
                              "warp_voxel_pairs": float(np.mean([s["warp_voxel_pairs"] for s in stats]))},
            "train_iteration": {"what": "step + svr_adam_step (zero_grad) over raw and sh; outside `value`",
                                "ms": ms_iter / args.steps, "iterations_per_s": args.steps * world / (ms_iter * 1e-3)}}

    # ---- NEXT-1 (not part of `value`): one depth-quantile pruning step on the w_max the steps above gathered, and the
    # compaction of the voxel arrays by its keep mask; HBM-bound streaming kernels, timed with CUDA events ----
    if rank == 0:
        po = pkg.SvrPruneOpts(8, 0.10, 0.05, 0.5, 0.3, 0.7, 1.0, 0.5, 0.05)
        ema = torch.zeros(sc.n, dtype=torch.float32, device=dev)
        st8 = torch.zeros(sc.n, dtype=torch.uint8, device=dev)
        keep = None
        for _ in range(2):
            keep, tau, n_removed = ctx.svr_prune_step(vox, ccams, w_max, ema, st8, po)
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        reps = 5
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(reps):
                keep, tau, n_removed = ctx.svr_prune_step(vox, ccams, w_max, ema, st8, po)
            e1.record(stream)
            for _ in range(reps):
                for arr in (vox.ijkl, vox.raw, vox.sh):
                    ctx.svr_compact_rows(keep, arr)
            e2.record(stream)
        torch.cuda.synchronize()
        ms_prune, ms_compact = e0.elapsed_time(e1) / reps, e1.elapsed_time(e2) / reps
        row_bytes = 8 + 32 + 12 * sc.n_basis
        kept = int(keep.sum().item())
        prune_bytes = sc.n * (8 + 4 + 4 + 4 + 1 + 1 + 1)             # ijkl, w_max, ema r/w, state r/w, keep
        compact_bytes = sc.n * (1 + row_bytes) + kept * row_bytes     # keep + all rows read, kept rows written
        line["next1_prune"] = {
            "what": "svr_prune_step (P:143-172, 8 depth bins, all cameras) + svr_compact_rows(ijkl, raw, sh); outside `value`",
            "prune_ms": ms_prune, "compact_ms": ms_compact, "removed": int(n_removed), "kept": kept,
            "prune_roofline": {"bound": "hbm", "achieved": prune_bytes / (ms_prune * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                               "frac": prune_bytes / (ms_prune * 1e-3) / 1e9 / peaks["hbm_gbs"],
                               "algorithmic": "23 B per voxel (ijkl, w_max, ema r/w, state r/w, keep)"},
            "compact_roofline": {"bound": "hbm", "achieved": compact_bytes / (ms_compact * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                                 "unit": "GB/s", "frac": compact_bytes / (ms_compact * 1e-3) / 1e9 / peaks["hbm_gbs"]}}

        # NEXT-2: priority-driven subdivision: selection (usefulness = w_max) and the 1 -> 8 split of 1% of the voxels
        so = pkg.SvrSubdivOpts(1.0, 0.2, sc.max_level, sc.n // 100, 1, 0.0, 0.0)
        split, _, _, n_split = ctx.svr_subdivide_select(vox, ccams, w_max, so)
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(reps):
                split, _, _, n_split = ctx.svr_subdivide_select(vox, ccams, w_max, so)
            e1.record(stream)
            for _ in range(reps):
                ctx.svr_subdivide_apply(vox, split, n_split)
            e2.record(stream)
        torch.cuda.synchronize()
        ms_sel, ms_app = e0.elapsed_time(e1) / reps, e1.elapsed_time(e2) / reps
        app_bytes = sc.n * (1 + row_bytes) + (sc.n + 7 * n_split) * row_bytes
        line["next2_subdivide"] = {
            "what": "svr_subdivide_select (eqs. 13-16, budget = 1% of the voxels) + svr_subdivide_apply (1 -> 8); outside `value`",
            "select_ms": ms_sel, "apply_ms": ms_app, "n_split": int(n_split),
            "apply_roofline": {"bound": "hbm", "achieved": app_bytes / (ms_app * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                               "frac": app_bytes / (ms_app * 1e-3) / 1e9 / peaks["hbm_gbs"]}}

        # NEXT-4 (part): fused Adam over the SH coefficients (the largest parameter tensor), gradient cleared in the same pass
        theta = vox.sh.view(-1)
        gflat, m1, v1 = g_sh.view(-1), torch.zeros_like(theta), torch.zeros_like(theta)
        ctx.svr_adam_step(theta, gflat, m1, v1, 0.0, 0.9, 0.999, 1e-8, 1, zero_grad=True)      # lr = 0: parameters unchanged
        e0, e1 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
        with torch.cuda.stream(stream):
            e0.record(stream)
            for k in range(reps):
                ctx.svr_adam_step(theta, gflat, m1, v1, 0.0, 0.9, 0.999, 1e-8, 2 + k, zero_grad=True)
            e1.record(stream)
        torch.cuda.synchronize()
        ms_adam = e0.elapsed_time(e1) / reps
        adam_bytes = theta.numel() * 32
        line["next4_adam"] = {"what": "svr_adam_step over sh [n,16,3] with zero_grad (32 B per parameter); outside `value`",
                              "ms": ms_adam, "params": int(theta.numel()),
                              "roofline": {"bound": "hbm", "achieved": adam_bytes / (ms_adam * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                                           "unit": "GB/s", "frac": adam_bytes / (ms_adam * 1e-3) / 1e9 / peaks["hbm_gbs"]}}

        # NEXT-4 (part): L_tv over the raw corner densities, gradient accumulated into g_raw
        lt = torch.empty(1, dtype=torch.float32, device=dev)
        ctx.svr_tv_loss_grad(vox.raw, g_raw, 1e-3, loss=lt)
        e0, e1 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(reps):
                ctx.svr_tv_loss_grad(vox.raw, g_raw, 1e-3, loss=lt)
            e1.record(stream)
        torch.cuda.synchronize()
        ms_tv = e0.elapsed_time(e1) / reps
        tv_bytes = sc.n * 96
        line["next4_tv"] = {"what": "svr_tv_loss_grad over raw [n,8] (32 B read + 64 B read-modify-write per voxel); outside `value`",
                            "ms": ms_tv, "L_tv": float(lt.item()),
                            "roofline": {"bound": "hbm", "achieved": tv_bytes / (ms_tv * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                                         "unit": "GB/s", "frac": tv_bytes / (ms_tv * 1e-3) / 1e9 / peaks["hbm_gbs"]}}

        # NEXT-3 (part): L_SSIM and its gradient on the last render against its target, accumulated onto dL
        ls = torch.empty(1, dtype=torch.float32, device=dev)
        ctx.svr_ssim_loss_grad(image, targets[0], 0.2, dL=dL, loss=ls, accumulate=True)
        e0, e1 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(reps):
                ctx.svr_ssim_loss_grad(image, targets[0], 0.2, dL=dL, loss=ls, accumulate=True)
            e1.record(stream)
        torch.cuda.synchronize()
        ms_ssim = e0.elapsed_time(e1) / reps
        ssim_bytes = H * W * 48          # algorithmic: render, target, dL read + dL written, 12 B each per pixel (the kernels move 132 B)
        line["next3_ssim"] = {"what": "svr_ssim_loss_grad (eq. 17 L_SSIM, 11-tap Gaussian window) accumulated onto dL; outside `value`",
                              "ms": ms_ssim, "L_ssim": float(ls.item()),
                              "roofline": {"bound": "hbm", "achieved": ssim_bytes / (ms_ssim * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                                           "unit": "GB/s", "frac": ssim_bytes / (ms_ssim * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                           "algorithmic": "48 B per pixel"}}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        n_rays = args.cpu_baseline_rays
        dt = oracle_sample_run(cfg, cams[0], n_rays, 4242)
        # every oracle call first bins the voxels and evaluates the per-view colours of all of them, whatever the number of
        # rays: timed on its own with a one-ray sample, so that the sample-size dependence of `value` can be read off
        dt_setup = oracle_sample_run(cfg, cams[0], 1, 4243)
        line["cpu_baseline"] = {"value": n_rays / dt / 1e6, "unit": "Mrays/s", "cores": oracle.num_threads(), "kind": "oracle",
                                "sample": f"{n_rays} seeded rays of camera 0 (of {rays}), bucketed fp64 oracle, forward+backward, "
                                          f"{dt:.1f} s of which {dt_setup:.1f} s are the per-call set-up (binning + per-view colours of all "
                                          f"voxels, independent of the ray count)",
                                "setup_s": dt_setup,
                                "value_excluding_setup": n_rays / max(dt - dt_setup, 1e-9) / 1e6}
    # last keys of the line (the driver's record keeps the tail): the rest of BASELINE.json's metric
    line["stage_ms_per_step"] = stage_ms
    line["peak_vram_bytes"] = peak_vram
    line["render_fps"] = line.pop("render_fps")
    if rank == 0:
        print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
