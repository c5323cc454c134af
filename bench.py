#!/usr/bin/env python
"""bench.py -- ICM iterations/s of the KCS hot path on B200 (BASELINE.json `metric`), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--impl ours|reference] [--no-sweeps]

A "step" is one pass of the whole hot path = one `kcs_icm_iteration` (kinetic model curve -> S x (forward
projection, Poisson ratio, back-projection, OSL update) -> n_lm MAP-LM steps) on the seeded synthetic workload
(kcs_inputs).  Default workload: C2 = BASELINE.json configs[1].

  value      whole-job ICM iterations/s with y, r, x, theta, lambda resident in HBM (CUDA events on the launch stream,
             L2 flushed between steps, max over ranks).
  e2e        the same through kcs_icm_run_host with pinned HOST buffers: H2D of y, r, x, theta, lambda and D2H of
             x, theta, lambda inside the timed region.
  roofline   the dominant kernel class of the step (per-kernel CUDA events from kcs_profile_*, a second pass of K
             steps): algorithmic flops / mean launch time against the FP32 FMA peak derived from
             the SM count and clocks.max.sm (74.4 TFLOP/s); the FP32, FP64, L2 and L1 peaks measured in the same run by
             kcs_probe_peak are printed beside it (`peaks_measured`).
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on this box's host cores, one ICM iteration of the same workload.
  sweeps     C5(a)/(b) kernel sweeps on the C4 geometry (projector Gsamples/s by frames per launch, MAP-LM fits/s by
             gamma) and one C4 ICM iteration, unless --no-sweeps.

N > 1 (torchrun): the path does not shard (BASELINE north_star: one GPU) -> N independent replicas, no collective
on the data path; value = N x iterations / max-over-ranks time ("replicas only").
--impl reference: the oracle timed on the host cores (rank 0 only), same metric / config.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import kcs_inputs as ki  # noqa: E402

METRIC = "ICM iterations/s"
UNIT = "it/s"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples: " + " | ".join(",".join(r) for r in self.rows[:2])]}
        load = [c for c, w in zip(sm, pw) if w >= 0.5 * max(pw)] or sm  # samples taken while the GPU was busy
        return {"sm_mhz": float(np.median(load)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "samples_under_load": len(load), "reasons": sorted(reasons),
                "window": "warm-up + timed steps + per-kernel pass"}


# ------------------------------------------------------------------------------------------------ workload
def flops_model(cfg: dict) -> dict:
    """Algorithmic work per launch of each kernel class."""
    T, nz, ny, nx = cfg["n_frames"], cfg["nz"], cfg["ny"], cfg["nx"]
    A, B, K, S = cfg["n_angles"], cfg["n_bins"], cfg["n_steps"], cfg["n_subsets"]
    sf_sub = T * nz * (A // S) * B * K        # sample-frames of one subset forward projection
    vaf_sub = T * nz * ny * nx * (A // S)     # voxel-angle-frames of one subset back-projection
    return {
        # 4 taps x 1 FMA; every tap is a 4-byte read through L1 (16 B), every pixel-frame comes from L2 once per angle (4 B)
        "forward": {"units": sf_sub, "flop_per_unit": 8.0, "l2_bytes_per_unit": 4.0, "l1_bytes_per_unit": 16.0},
        # 3 merged bins x 1 FMA; the 2x2 block's 5-bin window is 5 lines per 4 voxels (5 B), ~0.4 B of it new from L2
        "back": {"units": vaf_sub, "flop_per_unit": 6.0, "l2_bytes_per_unit": 0.4, "l1_bytes_per_unit": 5.0},
    }


def build_problem(ctx, cfg, torch, noisy=True):
    """Seeded synthetic workload; the forward model used to make the data is the CUDA library's (bench never takes a
    value from the oracle)."""
    T, nz, ny, nx, A, B = cfg["n_frames"], cfg["nz"], cfg["ny"], cfg["nx"], cfg["n_angles"], cfg["n_bins"]
    dev = torch.device("cuda", torch.cuda.current_device())

    def kin(theta):
        th = torch.tensor(np.asarray(theta), dtype=torch.float32, device=dev).contiguous()
        F = torch.zeros((T, nz, ny, nx), dtype=torch.float32, device=dev)
        ctx.kinetic_eval(th, F)
        return F.cpu().numpy().astype(np.float64)

    def fwd(x):
        x = np.asarray(x)
        nf = x.shape[0]
        xd = torch.zeros((T, nz, ny, nx), dtype=torch.float32, device=dev)
        xd[:nf] = torch.tensor(x, dtype=torch.float32, device=dev)
        yd = torch.zeros((T, nz, A, B), dtype=torch.float32, device=dev)
        ctx.forward_project(xd, yd, -1, 0, nf)
        return yd[:nf].cpu().numpy().astype(np.float64)

    mask = ctx.mask()
    prob = ki.make_problem(cfg, mask, kin, fwd, noisy=noisy)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], fwd)
    return mask, prob, (x0, th0, lam0)


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def max_over_ranks(seconds: float, dist, device) -> float:
    """Replicas only: the job's time is the slowest rank's; no collective touches the data path."""
    if dist is None:
        return seconds
    import torch
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_throughput(world: int, steps: int, seconds: float) -> float:
    """Whole-job ICM iterations/s of `world` independent replicas that each ran `steps` iterations in `seconds` (max)."""
    return world * steps / seconds


def load_traffic(workload: str, cls: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
    `ncu --set full` capture (profiles/traffic.csv: workload,kernel_class,dram_bytes_per_launch), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(p) as f:
            for line in f:
                c = [t.strip() for t in line.split(",")]
                if len(c) >= 3 and c[0] == workload and c[1] == cls:
                    return float(c[2])
    except Exception:
        pass
    return None


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import paper_1803_10045_b200 as kcs

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = ki.config(args.workload)
    ctx = kcs.Context(cfg)
    T, nz, ny, nx, A, B = cfg["n_frames"], cfg["nz"], cfg["ny"], cfg["nx"], cfg["n_angles"], cfg["n_bins"]
    t0 = time.time()
    mask, prob, (x0, th0, lam0) = build_problem(ctx, cfg, torch)
    log(f"[bench] rank {rank}: workload {args.workload} built in {time.time() - t0:.1f} s "
        f"(scale {prob['scale']:.4g}, counts {prob['y'].sum():.4g})")
    f32 = lambda a: torch.tensor(np.asarray(a), dtype=torch.float32, device=dev).contiguous()
    y, r = f32(prob["y"]), f32(prob["r"])
    x0d, th0d, lam0d = f32(x0), f32(th0), f32(lam0)
    x, th, lam = x0d.clone(), th0d.clone(), lam0d.clone()
    scale = float(prob["scale"])
    n_icm = cfg["n_icm"]
    flush = torch.empty(96 * 1024 * 1024, dtype=torch.float32, device=dev)  # 384 MB > 126 MB L2

    def reset():
        x.copy_(x0d); th.copy_(th0d); lam.copy_(lam0d)

    def step(i):
        """ICM iteration (i mod n_icm) + 1 of a reconstruction that restarts every n_icm steps (Q17: beta = 0 first)."""
        if i % n_icm == 0:
            reset()
        flush.zero_()  # evict the previous step's data from L2 (outside the event pair)
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.icm_iteration(y, r, scale, x, th, lam, 0.0 if i % n_icm == 0 else cfg["beta"], cfg["gamma"], cfg["delta"],
                          cfg["n_lm"])
        e1.record()
        return e0, e1

    # nvidia-smi polls at >= 100 ms: sample from the warm-up to the end of the per-kernel pass (same steps throughout)
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
        time.sleep(0.3)
    for i in range(args.warmup):
        step(i)
    barrier()
    n0 = ctx.launch_count()
    evs = [step(i) for i in range(args.steps)]
    barrier()
    launches = ctx.launch_count() - n0
    ms_total = float(sum(a.elapsed_time(b) for a, b in evs))
    ms_total = max_over_ranks(ms_total, dist, dev)
    ms_per_step = ms_total / args.steps
    value = replica_throughput(world, args.steps, ms_total * 1e-3)

    # ---- per-kernel pass (same steps again, profiling events on) -> roofline of the dominant kernel
    ctx.profile_enable(True)
    ctx.profile_read()
    pevs = [step(i) for i in range(args.steps)]
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    torch.cuda.synchronize()
    clk = clocks.stop() if rank == 0 else None
    ms_prof = float(sum(a.elapsed_time(b) for a, b in pevs)) / args.steps
    per_class = {k: {"ms_per_step": v[0] / args.steps, "launches_per_step": v[1] / args.steps} for k, v in prof.items() if v[1]}
    fm = flops_model(cfg)
    dom = max((k for k in per_class if k in fm), key=lambda k: per_class[k]["ms_per_step"])
    dom_ms = prof[dom][0] / prof[dom][1]
    peak_fp32_derived = 148 * 128 * 2 * 1.965e9 * 1e-12  # SMs x FP32 lanes x 2 x clocks.max.sm
    achieved = fm[dom]["units"] * fm[dom]["flop_per_unit"] / (dom_ms * 1e-3) * 1e-12
    roofline = {"bound": "alu", "kernel": {"forward": "k_forward (projector + Poisson ratio)",
                                           "back": "k_back (gather back-projector + OSL)"}[dom],
                "achieved": achieved, "peak": peak_fp32_derived, "unit": "TFLOP/s", "frac": achieved / peak_fp32_derived,
                "traffic": load_traffic(args.workload, dom), "avg_launch_ms": dom_ms,
                "units_per_launch": fm[dom]["units"], "flop_per_unit": fm[dom]["flop_per_unit"],
                "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (no FP32 figure in MEASURED_PEAKS.json)",
                "share_of_step": per_class[dom]["ms_per_step"] / ms_prof}
    result = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 (projector, OSL, storage) + f64 (kinetic model, MAP-LM registers)", "data": "synthetic",
        "config": {"workload": args.workload, "image": [nx, ny, nz], "sinogram": [A, B], "frames": T,
                   "subsets": cfg["n_subsets"], "n_lm": cfg["n_lm"], "l2": "flushed between steps (384 MB write)",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "gpu_launches": int(launches), "clocks": clk, "roofline": roofline,
        "kernels": per_class, "ms_per_step_profiled": ms_prof,
    }
    if rank == 0 and world == 1:
        try:
            result["peaks_measured"] = {k: ctx.probe_peak(k) for k in kcs.PEAK_PROBES}
            roofline["peak_measured_fp32_tflops"] = result["peaks_measured"]["fp32_tflops"]
            roofline["l2_achieved_gbs"] = fm[dom]["units"] * fm[dom]["l2_bytes_per_unit"] / (dom_ms * 1e-3) * 1e-9
            # the unit that actually binds the projector pair: L1 data-pipe bytes against the L1 probe
            roofline["l1_achieved_gbs"] = fm[dom]["units"] * fm[dom]["l1_bytes_per_unit"] / (dom_ms * 1e-3) * 1e-9
            roofline["l1_frac_of_measured"] = roofline["l1_achieved_gbs"] / result["peaks_measured"]["l1_gbs"]
        except Exception as e:  # a probe failure must not lose the bench line
            result["peaks_measured"] = {"error": str(e)}

    # ---- end to end through the host-buffer entry point
    result["e2e"] = run_e2e(ctx, cfg, prob, (x0, th0, lam0), torch, args, world, dist, dev, flush)
    if rank == 0 and world == 1:
        result["cpu_baseline"] = cpu_baseline(cfg, args.workload)
        if not args.no_sweeps:
            ctx.close()
            del y, x, th, lam, x0d, th0d
            torch.cuda.empty_cache()
            try:
                result["sweeps"] = run_sweeps(torch, kcs, dev)
            except Exception as e:
                result["sweeps"] = {"error": repr(e)}
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(result), flush=True)


def run_e2e(ctx, cfg, prob, state0, torch, args, world, dist, dev, flush):
    """kcs_icm_run_host with pinned host buffers: H2D (y, r, x, theta, lambda) and D2H (x, theta, lambda) every step."""
    x0, th0, lam0 = state0
    pin = lambda a: torch.tensor(np.asarray(a), dtype=torch.float32).contiguous().pin_memory()
    hy, hr = pin(prob["y"]), pin(prob["r"])
    hx, hth, hlam = pin(x0), pin(th0), pin(lam0)
    scale, n_icm = float(prob["scale"]), cfg["n_icm"]

    def one(i):
        if i % n_icm == 0:
            hx.copy_(torch.tensor(x0, dtype=torch.float32)); hth.copy_(torch.tensor(th0, dtype=torch.float32)); hlam.zero_()
        flush.zero_()
        torch.cuda.synchronize()
        t = time.perf_counter()
        b = 0.0 if i % n_icm == 0 else cfg["beta"]
        ctx.icm_run_host(hy, hr, scale, hx, hth, hlam, b, b, cfg["gamma"], cfg["delta"], cfg["n_lm"], 1)  # synchronous
        return time.perf_counter() - t

    for i in range(args.warmup):
        one(i)
    if dist is not None:
        dist.barrier()
    tot = sum(one(i) for i in range(args.steps))
    tot = max_over_ranks(tot, dist, dev)
    h2d = 4 * (hy.numel() + hr.numel() + hx.numel() + hth.numel() + hlam.numel())
    d2h = 4 * (hx.numel() + hth.numel() + hlam.numel())
    return {"value": replica_throughput(world, args.steps, tot), "unit": UNIT, "ms_per_step": 1e3 * tot / args.steps,
            "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
            "api": "kcs_icm_run_host (n_iter = 1), pinned host buffers, wall clock around the synchronous call"}


# ------------------------------------------------------------------------------------------------ oracle legs
def oracle_sample(cfg: dict, workload: str):
    """A bounded sample of the workload for the oracle: the first nz_s slices (slices are independent direct planes
    in the OS pass and the LM cost is per voxel), with counts scaled by nz_s / nz."""
    nz_s = {"C1": 1, "C2": 2, "C3": 2, "C4": 1, "C5": 1}.get(workload, 1)
    nz_s = min(nz_s, cfg["nz"])
    sub = dict(cfg, nz=nz_s, counts=cfg["counts"] * nz_s / cfg["nz"])  # 3-D phantoms: the central nz_s slices
    return sub, nz_s


def oracle_problem(workload: str):
    from oracle import Oracle
    cfg = ki.config(workload)
    sub, nz_s = oracle_sample(cfg, workload)
    o = Oracle(sub)
    mask = o.default_mask()
    prob = ki.make_problem(sub, mask, o.kinetic_eval, o.forward_project, noisy=True)
    st = ki.initial_state(sub, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    return cfg, sub, nz_s, o, prob, st


def cpu_baseline(cfg: dict, workload: str) -> dict:
    """The oracle as it stands, one ICM iteration (beta = 0, the first of a reconstruction) on the bounded sample."""
    from oracle import Oracle
    _, sub, nz_s, o, prob, (x0, th0, lam0) = oracle_problem(workload)
    t = time.perf_counter()
    o.icm_iteration(prob["y"], prob["r"], prob["scale"], x0, th0, lam0, 0.0, sub["gamma"], sub["delta"], sub["n_lm"])
    dt = time.perf_counter() - t
    return {"value": (nz_s / cfg["nz"]) / dt, "unit": UNIT, "cores": Oracle.num_threads(), "kind": "oracle",
            "sample": f"one ICM iteration on {nz_s} of {cfg['nz']} slices of {workload} ({dt:.2f} s), scaled by {nz_s}/{cfg['nz']}",
            "seconds": dt}


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return
    from oracle import Oracle
    cfg, sub, nz_s, o, prob, (x0, th0, lam0) = oracle_problem(args.workload)
    x, th, lam = x0, th0, lam0
    n_icm = sub["n_icm"]

    def one(i):
        nonlocal x, th, lam
        if i % n_icm == 0:
            x, th, lam = x0, th0, lam0
        t = time.perf_counter()
        x, th, lam = o.icm_iteration(prob["y"], prob["r"], prob["scale"], x, th, lam, 0.0 if i % n_icm == 0 else sub["beta"],
                                     sub["gamma"], sub["delta"], sub["n_lm"])
        return time.perf_counter() - t

    for i in range(args.warmup):
        one(i)
    tot = sum(one(i) for i in range(args.steps))
    value = (nz_s / cfg["nz"]) * args.steps / tot
    sample = f"each step = one ICM iteration on {nz_s} of {cfg['nz']} slices of {args.workload}, scaled by {nz_s}/{cfg['nz']}"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "image": [cfg["nx"], cfg["ny"], cfg["nz"]],
                   "sinogram": [cfg["n_angles"], cfg["n_bins"]], "frames": cfg["n_frames"], "subsets": cfg["n_subsets"],
                   "n_lm": cfg["n_lm"], "parallelism": "host cores (OpenMP)"},
        "gpu_launches": 0,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": Oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


# ------------------------------------------------------------------------------------------------ C5 sweeps
def run_sweeps(torch, kcs, dev) -> dict:
    """BASELINE configs[4] (C5) on the C4 geometry, plus one C4 ICM iteration.  Inputs are made on the device
    (noiseless activity from the C4 phantom; Poisson data from torch's seeded generator) -- throughput only."""
    out = {}
    cfg = ki.config("C5")
    T, nz, ny, nx, A, B, K = cfg["n_frames"], cfg["nz"], cfg["ny"], cfg["nx"], cfg["n_angles"], cfg["n_bins"], cfg["n_steps"]
    ctx = kcs.Context(cfg)
    mask = ctx.mask()
    md = torch.tensor(mask, dtype=torch.float32, device=dev)
    _, th_true = ki.phantom(cfg)
    th_true = torch.tensor(th_true, dtype=torch.float32, device=dev) * md[None, None]
    x = torch.zeros((T, nz, ny, nx), dtype=torch.float32, device=dev)
    ctx.kinetic_eval(th_true.contiguous(), x)
    x *= md[None, None]
    y = torch.zeros((T, nz, A, B), dtype=torch.float32, device=dev)
    b = torch.zeros_like(x)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(fn, reps=2):
        fn()  # warm-up
        torch.cuda.synchronize()
        best = 1e30
        for _ in range(reps):
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        return best

    # (a) projector pair alone, frames batched per launch nf in {1, 4, 12, 29}; inputs (1.7 GB + 1.3 GB) exceed L2
    sf = float(T) * nz * A * B * K
    out["projector"] = []
    ctx.profile_enable(True)
    for nf in (1, 4, 12, 29):
        chunks = [(f0, min(nf, T - f0)) for f0 in range(0, T, nf)]
        ctx.profile_read()
        ms_f = timed(lambda: [ctx.forward_project(x, y, -1, f0, n) for f0, n in chunks], reps=1)
        pf = ctx.profile_read()
        ms_b = timed(lambda: [ctx.back_project(y, b, -1, f0, n) for f0, n in chunks], reps=1)
        pb = ctx.profile_read()
        out["projector"].append({
            "frames_per_launch": nf, "launches": len(chunks),
            "forward_ms": ms_f, "forward_gsamples_s": sf / ms_f * 1e-6, "forward_kernel_ms": pf["forward"][0] / 2,
            "back_ms": ms_b, "back_gsamples_s": sf / ms_b * 1e-6, "back_kernel_ms": pb["back"][0] / 2})
    ctx.profile_enable(False)
    # (b) MAP-LM alone, 20 steps, start within +/-50 % of the truth, gamma in {0, 0.05, 0.5}
    rng = torch.Generator(device=dev)
    rng.manual_seed(4)
    start = (th_true * (0.5 + torch.rand(th_true.shape, generator=rng, device=dev))).contiguous()
    nfit = float(mask.sum()) * nz
    out["map_lm"] = []
    for gamma in (0.0, 0.05, 0.5):
        def fit():
            th = start.clone()
            lam = torch.zeros((nz, ny, nx), dtype=torch.float32, device=dev)
            ctx.map_lm(x, th, lam, gamma, cfg["delta"], 20)
        th_w = start.clone(); lam_w = torch.zeros((nz, ny, nx), dtype=torch.float32, device=dev)
        ctx.map_lm(x, th_w, lam_w, gamma, cfg["delta"], 20)  # warm-up
        torch.cuda.synchronize()
        th = start.clone(); lam = torch.zeros_like(lam_w)
        e0.record(); ctx.map_lm(x, th, lam, gamma, cfg["delta"], 20); e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        out["map_lm"].append({"gamma": gamma, "steps": 20, "ms": ms, "fits_s": nfit / ms * 1e3,
                              "voxel_steps_s": nfit * 20 / ms * 1e3})
    # one C4 ICM iteration (noisy data, 2e8 counts, randoms 10 %)
    ctx.forward_project(x, y)
    scale = cfg["counts"] / float(y.sum(dtype=torch.float64))
    r = (0.1 * scale * y.reshape(T, -1).mean(dim=1, dtype=torch.float64)).float().contiguous()
    y.mul_(scale).add_(r[:, None, None, None])
    torch.manual_seed(1003)
    yn = torch.poisson(y)
    x0 = (x.reshape(T, -1).sum(1) / (md.sum() * nz))[:, None, None, None] * md[None, None].expand(1, nz, ny, nx)
    x0 = x0.contiguous()
    th0 = (torch.tensor(ki.THETA0, dtype=torch.float32, device=dev)[:, None, None, None] * md[None, None].expand(1, nz, ny, nx)).contiguous()
    lam = torch.zeros((nz, ny, nx), dtype=torch.float32, device=dev)
    xx, tt = x0.clone(), th0.clone()
    ctx.icm_iteration(yn, r, scale, xx, tt, lam, 0.0, cfg["gamma"], cfg["delta"], cfg["n_lm"])  # iteration 1 (warm-up)
    torch.cuda.synchronize()
    ms = []
    for _ in range(3):
        e0.record()
        ctx.icm_iteration(yn, r, scale, xx, tt, lam, cfg["beta"], cfg["gamma"], cfg["delta"], cfg["n_lm"])
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    out["icm_C4"] = {"ms_per_iteration": float(np.median(ms)), "it_s": 1e3 / float(np.median(ms)),
                     "finite": bool(torch.isfinite(xx).all() and torch.isfinite(tt).all())}
    ctx.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="C2", choices=["C1", "C2", "C3", "C4"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweeps", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
