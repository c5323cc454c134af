#!/usr/bin/env python
"""bench.py -- ICM iterations/s of the KCS hot path on B200 (BASELINE.json `metric`), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl ours|reference] [--no-sweeps]
                    [--no-per-config]

A "step" is one pass of the whole hot path = one ICM iteration (kinetic model curve -> S x (forward projection,
Poisson ratio, back-projection, OSL update) -> n_lm MAP-LM steps) on the seeded synthetic
workload (kcs_inputs).  Default workload: C4 = BASELINE.json configs[3], the largest
single-GPU configuration (BASELINE's `metric` names no config).

  value      whole-job ICM iterations/s with y, r, x, theta, lambda resident in HBM, CUDA events on the launch stream,
             max over ranks.  C3 / C4 (inputs of 0.3 / 3.3 GB, larger than the 126 MB L2): the K steps are run as
             reconstructions of n_icm = 10 iterations through kcs_icm_run (the ICM loop of P:118-125; y is packed once
             per reconstruction); C1 / C2 (inputs fit in L2): one kcs_icm_iteration per step with L2 flushed
             between steps.  `config.l2` says which.
  e2e        the same metric through kcs_icm_run_host with pinned HOST buffers: H2D of y, r, x, theta, lambda and D2H
             of x, theta, lambda inside the timed region of every step.
  roofline   the dominant kernel class of the step (per-kernel CUDA events from kcs_profile_*, a second pass of the
             same K steps, every kernel launched over the whole volume on one stream).  SURVEY.md 8(d): T_lb = max(HBM bytes / BW_HBM, L2 bytes / BW_L2, flops / P_FP32); `bound`
             names the largest term, frac = T_lb / measured launch time; achieved / peak are that term's.  All three
             terms, for every kernel class, are under `roofline.classes`.  BW_HBM = MEASURED_PEAKS.json; BW_L2 and
             P_FP32 / P_FP64 are measured in this run by libkcs_probe.so (include/kcs_probe.h).  Units are the EXECUTED
             ones (rays clipped to the field of view, in-mask voxels); the defined operation's count is printed too.
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on this box's host cores: one ICM iteration of a bounded
             sample (a few slices) of the same workload.
  per_config ICM it/s of the other configurations (C1, C2, C3) and of C1 as one batch of 100 noise realisations
             (kcs_config.n_replicas), unless --no-per-config.
  sweeps     C5(a)/(b) kernel sweeps on the C4 geometry (projector Gsamples/s by frames per launch, MAP-LM fits/s by
             gamma), each with its roofline fraction, unless --no-sweeps.

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
L2_BYTES = 126e6
HBM_FALLBACK_GBS = 6500.0  # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


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


# ------------------------------------------------------------------------------------------------ work model
def lm_flops_per_eval(T: int) -> float:
    """Model + Jacobian + normal equations of one voxel, counted from the formulas of DESIGN.md section 6 (one flop per
    add / multiply, 2 per FMA): 92 per frame (frame recursion 7, G and dG/da at the frame end 30, F and its four
    derivatives 23, J^T J / J^T r / Phi accumulation 32) + 300 per voxel (rate scalars, one expm1 and one E1 series per
    distinct frame duration)."""
    return 92.0 * T + 300.0


def lm_flops_per_step(T: int) -> float:
    """One LM step after the first of a call: one evaluation + Cholesky solve, Huber sums, accept test (~500)."""
    return lm_flops_per_eval(T) + 500.0


def fwd_executed_samples_per_ray_row(cfg: dict, mask: np.ndarray) -> float:
    """Sum over the bins of one sinogram row of the samples k_forward executes in the ICM path, where rays are clipped to
    the field-of-view circle (mask radius + 1.5 voxels; x is zero outside the mask)."""
    nx, ny, B, K = cfg["nx"], cfg["ny"], cfg["n_bins"], cfg["n_steps"]
    jj, ii = np.nonzero(mask)
    X, Y = (ii - 0.5 * (nx - 1)) * cfg["vx"], (jj - 0.5 * (ny - 1)) * cfg["vy"]
    rc = np.sqrt((X * X + Y * Y).max()) + 1.5 * max(cfg["vx"], cfg["vy"])
    s = (np.arange(B) - 0.5 * (B - 1)) * cfg["bin_mm"]
    h2 = rc * rc - s * s
    h = np.sqrt(np.maximum(h2, 0.0)) / cfg["step_mm"]
    ck = 0.5 * (K - 1)
    n = np.floor(np.minimum(K - 1, ck + h)) - np.ceil(np.maximum(0.0, ck - h)) + 1
    return float(np.where(h2 >= 0, np.maximum(n, 0), 0).sum())


def work_model(cfg: dict, mask: np.ndarray, T: int | None = None, subset: bool = True, clipped: bool = True) -> dict:
    """Algorithmic work PER LAUNCH of each kernel class.  `executed` counts what
    the ICM path runs (FOV-clipped rays, in-mask voxels); `defined` the full operation T x rays x steps."""
    T = cfg["n_frames"] if T is None else T
    nz, ny, nx = cfg["nz"], cfg["ny"], cfg["nx"]
    A, B, K, S = cfg["n_angles"], cfg["n_bins"], cfg["n_steps"], cfg["n_subsets"]
    As = A // S if subset else A
    n_in = int(mask.sum())
    rays = nz * As * B
    f_def = float(T) * rays * K
    f_exe = float(T) * nz * As * fwd_executed_samples_per_ray_row(cfg, mask) if clipped else f_def
    b_def = float(T) * nz * ny * nx * As
    b_exe = float(T) * nz * n_in * As if clipped else b_def
    vin = float(nz) * n_in
    return {
        # 4 taps x 1 FMA per sample-frame; every pixel-frame of a slice comes from L2 once per angle (4 B per sample-frame);
        # HBM: the in-FOV part of x once, y read and q written
        "forward": {"units": f_exe, "units_defined": f_def, "unit": "sample-frames", "flops": 8.0 * f_exe,
                    "l2_bytes": 4.0 * f_exe, "hbm_bytes": 4.0 * T * (vin + 2.0 * rays)},
        # <= 3 merged bin weights per voxel-angle-frame; 0.4 B of new sinogram data from L2 per unit (16x16-voxel tile);
        # HBM: q read, and for the fused OSL update x read + written and F read
        "back": {"units": b_exe, "units_defined": b_def, "unit": "voxel-angle-frames", "flops": 6.0 * b_exe,
                 "l2_bytes": 0.4 * b_exe, "hbm_bytes": 4.0 * T * (rays + (3.0 * vin if clipped else float(nz) * ny * nx))},
        # one LM step (not the first of a call): x_v read once (4T B), theta / lambda fp64 in + out, the 15 carried sums
        # in + out; neighbours come from L2 (6 x 4 x 8 B)
        "lm": {"units": vin, "units_defined": vin, "unit": "voxel-steps", "flops": lm_flops_per_step(T) * vin,
               "l2_bytes": 192.0 * vin, "hbm_bytes": (4.0 * T + 2 * 40.0 + 2 * 120.0) * vin},
    }


def bounds(w: dict, ms: float, peaks: dict) -> dict:
    """the three lower bounds of one launch, the binding one, and frac = T_lb / measured."""
    t = {"hbm": w["hbm_bytes"] / (peaks["hbm_gbs"] * 1e9) * 1e3,
         "l2": w["l2_bytes"] / (peaks["l2_gbs"] * 1e9) * 1e3,
         "alu": w["flops"] / (peaks["fp32_tflops"] * 1e12) * 1e3}
    bound = max(t, key=t.get)
    out = {"avg_launch_ms": ms, "bound": bound, "t_lb_ms": t[bound], "frac": t[bound] / ms, "t_bound_ms": t,
           "units": w["units"], "units_defined": w["units_defined"], "unit_name": w["unit"],
           "hbm_gbs": w["hbm_bytes"] / ms * 1e-6, "l2_gbs": w["l2_bytes"] / ms * 1e-6, "tflops": w["flops"] / ms * 1e-9,
           "units_per_s": w["units"] / ms * 1e3}
    return out


def measured_peaks(torch, kcs) -> dict:
    """HBM copy bandwidth from MEASURED_PEAKS.json (driver-written), the rest from libkcs_probe.so in this run."""
    p = {}
    try:
        mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        p["hbm_gbs"], p["hbm_source"] = float(mp["hbm_gbs"]), "MEASURED_PEAKS.json"
    except Exception:
        p["hbm_gbs"], p["hbm_source"] = HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md): MEASURED_PEAKS.json absent"
    for k in kcs.PEAK_PROBES:
        p[k] = kcs.probe_peak(k)
    # the L2 term of the projector pair is compared with the probe that has its access pattern (whole 128 B lines at
    # scattered addresses, L1 bypassed); the streaming figure is printed beside it
    p["l2_stream_gbs"] = p["l2_gbs"]
    p["l2_gbs"] = p["l2_gather_gbs"]
    p["source"] = "libkcs_probe.so in this run (fp32/fp64 FMA chains, L2 streaming, L2 line gather with ld.global.cg, L1 window)"
    return p


def load_traffic(workload: str, cls: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of a kernel class from the committed `ncu --set full`
    capture (profiles/traffic.csv: workload,kernel_class,dram_bytes_per_launch,capture), or (None, None)."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(p) as f:
            for line in f:
                c = [t.strip() for t in line.split(",")]
                if len(c) >= 3 and c[0] == workload and c[1] == cls:
                    return float(c[2]), (c[3] if len(c) > 3 else None)
    except Exception:
        pass
    return None, None


# ------------------------------------------------------------------------------------------------ workload
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


def input_bytes(cfg: dict) -> float:
    T = cfg["n_frames"]
    return 4.0 * T * (cfg["nz"] * cfg["ny"] * cfg["nx"] + cfg["nz"] * cfg["n_angles"] * cfg["n_bins"])


class IcmRunner:
    """Times K ICM iterations of one workload with the state resident in HBM.  Reconstructions restart every n_icm
    iterations from the Q17 start (beta = 0 in the first).  Inputs larger than L2: kcs_icm_run over whole
    reconstructions; else one kcs_icm_iteration per step with a 384 MB write between steps."""

    def __init__(self, torch, ctx, cfg, prob, state0, dev):
        self.torch, self.ctx, self.cfg = torch, ctx, cfg
        f32 = lambda a: torch.tensor(np.asarray(a), dtype=torch.float32, device=dev).contiguous()
        self.y, self.r = f32(prob["y"]), f32(prob["r"])
        self.x0, self.th0, self.lam0 = (f32(a) for a in state0)
        self.x, self.th, self.lam = self.x0.clone(), self.th0.clone(), self.lam0.clone()
        self.scale = float(prob["scale"])
        self.big = input_bytes(cfg) > L2_BYTES
        self.flush = None if self.big else torch.empty(96 * 1024 * 1024, dtype=torch.float32, device=dev)
        self.l2_note = ("inputs larger than L2 (%.2f GB), no flush; steps run as reconstructions of n_icm iterations "
                        "through kcs_icm_run" % (input_bytes(cfg) * 1e-9)) if self.big else \
            "flushed between steps (384 MB write), one kcs_icm_iteration per step"

    def reset(self):
        self.x.copy_(self.x0); self.th.copy_(self.th0); self.lam.copy_(self.lam0)

    def run(self, steps: int):
        """Enqueue `steps` iterations; returns the (start, end) event pairs that bracket the timed launches."""
        torch, ctx, cfg = self.torch, self.ctx, self.cfg
        n_icm, evs, i = cfg["n_icm"], [], 0
        while i < steps:
            self.reset()
            n = min(n_icm, steps - i)
            if self.big:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                ctx.icm_run(self.y, self.r, self.scale, self.x, self.th, self.lam, 0.0, cfg["beta"], cfg["gamma"],
                            cfg["delta"], cfg["n_lm"], n)
                e1.record()
                evs.append((e0, e1))
            else:
                for k in range(n):
                    self.flush.zero_()  # evict the previous step's data from L2 (outside the event pair)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    ctx.icm_iteration(self.y, self.r, self.scale, self.x, self.th, self.lam,
                                      0.0 if k == 0 else cfg["beta"], cfg["gamma"], cfg["delta"], cfg["n_lm"])
                    e1.record()
                    evs.append((e0, e1))
            i += n
        return evs


def time_config(torch, kcs, dev, name: str, steps: int, warmup: int) -> dict:
    """Resident ICM it/s of one configuration (per_config table)."""
    cfg = ki.config(name)
    ctx = kcs.Context(cfg)
    _, prob, st = build_problem(ctx, cfg, torch)
    run = IcmRunner(torch, ctx, cfg, prob, st, dev)
    run.run(warmup)
    torch.cuda.synchronize()
    n0 = ctx.launch_count()
    evs = run.run(steps)
    torch.cuda.synchronize()
    ms = float(sum(a.elapsed_time(b) for a, b in evs))
    out = {"it_s": steps / ms * 1e3, "ms_per_iteration": ms / steps, "steps": steps, "warmup": warmup,
           "gpu_launches_per_iteration": (ctx.launch_count() - n0) / steps, "l2": run.l2_note,
           "cuda_graph_replays": ctx.graph_replays(),
           "finite": bool(torch.isfinite(run.x).all() and torch.isfinite(run.th).all())}
    ctx.close()
    return out


def time_replicas(torch, kcs, dev, name: str, n_rep: int, steps: int, warmup: int) -> dict:
    """`n_rep` Poisson realisations of one small workload reconstructed in ONE batch
    (kcs_config.n_replicas): every launch covers n_rep x nz slices, so the launch-bound small configurations fill the GPU.
    Reports ICM iterations/s of the batch and replica-iterations/s."""
    base = ki.config(name)
    one = kcs.Context(base)
    _, prob, (x0, th0, lam0) = build_problem(one, base, torch, noisy=False)
    one.close()
    cfg = dict(base, n_replicas=n_rep)
    ctx = kcs.Context(cfg)
    batch = dict(prob, y=ki.noise_realisations(prob["ybar"], base["seed"], n_rep))
    st = (ki.tile_replicas(x0, 1, n_rep), ki.tile_replicas(th0, 1, n_rep), ki.tile_replicas(lam0, 0, n_rep))
    run = IcmRunner(torch, ctx, dict(cfg, nz=base["nz"] * n_rep), batch, st, dev)
    run.run(warmup)
    torch.cuda.synchronize()
    n0 = ctx.launch_count()
    evs = run.run(steps)
    torch.cuda.synchronize()
    ms = float(sum(a.elapsed_time(b) for a, b in evs))
    out = {"replicas": n_rep, "it_s": steps / ms * 1e3, "replica_it_s": n_rep * steps / ms * 1e3, "ms_per_iteration": ms / steps,
           "steps": steps, "warmup": warmup, "gpu_launches_per_iteration": (ctx.launch_count() - n0) / steps, "l2": run.l2_note,
           "finite": bool(torch.isfinite(run.x).all() and torch.isfinite(run.th).all())}
    ctx.close()
    return out


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import paper_1803_10045_b200 as kcs

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    # everything runs on one non-default stream: the legacy default stream cannot be captured, and the launch-bound
    # configurations (C1, C2) replay their iteration as a CUDA graph (kcs.h, kcs_use_graphs)
    torch.cuda.set_stream(torch.cuda.Stream(device=dev))
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
    mask, prob, state0 = build_problem(ctx, cfg, torch)
    log(f"[bench] rank {rank}: workload {args.workload} built in {time.time() - t0:.1f} s "
        f"(scale {prob['scale']:.4g}, counts {prob['y'].sum():.4g})")
    run = IcmRunner(torch, ctx, cfg, prob, state0, dev)

    # nvidia-smi polls at >= 100 ms: sample from the warm-up to the end of the per-kernel pass (same steps throughout)
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
        time.sleep(0.3)
    run.run(args.warmup)
    barrier()
    n0 = ctx.launch_count()
    evs = run.run(args.steps)
    barrier()
    launches = ctx.launch_count() - n0
    ms_total = float(sum(a.elapsed_time(b) for a, b in evs))
    ms_total = max_over_ranks(ms_total, dist, dev)
    ms_per_step = ms_total / args.steps
    value = replica_throughput(world, args.steps, ms_total * 1e-3)

    # ---- per-kernel pass (same steps again, profiling events on) -> per-class launch times
    ctx.profile_enable(True)
    ctx.profile_read()
    pevs = run.run(args.steps)
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    torch.cuda.synchronize()
    clk = clocks.stop() if rank == 0 else None
    ms_prof = float(sum(a.elapsed_time(b) for a, b in pevs)) / args.steps
    per_class = {k: {"ms_per_step": v[0] / args.steps, "launches_per_step": v[1] / args.steps} for k, v in prof.items() if v[1]}

    result = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 (projector, OSL, storage) + f64 (kinetic model, MAP-LM registers)", "data": "synthetic",
        "config": {"workload": args.workload, "image": [nx, ny, nz], "sinogram": [A, B], "frames": T,
                   "subsets": cfg["n_subsets"], "n_lm": cfg["n_lm"], "l2": run.l2_note,
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "gpu_launches": int(launches), "clocks": clk,
        "kernels": per_class, "ms_per_step_profiled": ms_prof,
    }
    peaks = None
    if rank == 0:
        try:
            peaks = measured_peaks(torch, kcs)
        except Exception as e:  # a probe failure must not lose the bench line
            peaks = {"error": repr(e), "hbm_gbs": HBM_FALLBACK_GBS, "l2_gbs": 17000.0, "fp32_tflops": 64.0, "fp64_tflops": 34.0}
        result["peaks_measured"] = peaks
        wm = work_model(cfg, mask)
        classes = {}
        for k in ("forward", "back", "lm"):
            if prof.get(k, (0, 0))[1]:
                classes[k] = bounds(wm[k], prof[k][0] / prof[k][1], peaks)
        if "lm" in classes:  # the fit runs on the FP64 pipe: its fraction of that pipe beside the FP32 target of BJ
            classes["lm"]["frac_of_fp64_peak"] = classes["lm"]["tflops"] / peaks["fp64_tflops"]
            classes["lm"]["frac_of_fp32_peak"] = classes["lm"]["tflops"] / peaks["fp32_tflops"]
        dom = max(classes, key=lambda k: per_class[k]["ms_per_step"])
        c = classes[dom]
        ach, pk, unit = {"hbm": (c["hbm_gbs"], peaks["hbm_gbs"], "GB/s"), "l2": (c["l2_gbs"], peaks["l2_gbs"], "GB/s"),
                         "alu": (c["tflops"], peaks["fp32_tflops"], "TFLOP/s")}[c["bound"]]
        traffic, capture = load_traffic(args.workload, dom)
        result["roofline"] = {
            "bound": c["bound"], "achieved": ach, "peak": pk, "unit": unit, "frac": c["frac"], "traffic": traffic,
            "traffic_capture": capture,
            "kernel": {"forward": "k_forward (projector + Poisson ratio)", "back": "k_back (gather back-projector + OSL)",
                       "lm": "k_lm_step (MAP-LM)"}[dom],
            "avg_launch_ms": c["avg_launch_ms"], "t_lb_ms": c["t_lb_ms"], "units_per_launch": c["units"],
            "units_defined_per_launch": c["units_defined"], "share_of_step": per_class[dom]["ms_per_step"] / ms_prof,
            "peak_source": {"hbm": peaks.get("hbm_source"), "l2": "L2 line-gather probe of this run (ld.global.cg)",
                            "alu": "FP32 FFMA probe of this run"}[c["bound"]],
            # the unit that physically binds the projector pair: L1 wavefronts, 16 B per sample-frame
            "l1_gbs": (16.0 if dom == "forward" else 5.0) * c["units"] / c["avg_launch_ms"] * 1e-6,
            "l1_peak_gbs": peaks.get("l1_gbs"),
            "step_t_lb_ms": sum(classes[k]["t_lb_ms"] * per_class[k]["launches_per_step"] for k in classes),
            "step_frac": sum(classes[k]["t_lb_ms"] * per_class[k]["launches_per_step"] for k in classes) / ms_per_step,
            "classes": classes,
            # kcs_icm_run splits the OS pass of a large volume in two z halves on two streams; with per-kernel timing on it
            # launches every kernel over the whole volume on one stream, so that the events bracket kernels running alone
            "profile_pass": "one stream, full-volume launches (timed steps: two z halves on two streams)",
        }

    # ---- end to end through the host-buffer entry point
    result["e2e"] = run_e2e(ctx, cfg, prob, state0, torch, args, world, dist, dev)
    ctx.close()
    del run
    torch.cuda.empty_cache()
    if rank == 0 and world == 1:
        result["cpu_baseline"] = cpu_baseline(cfg, args.workload)
        if not args.no_per_config:
            result["per_config"] = {args.workload: {"it_s": value, "ms_per_iteration": ms_per_step}}
            for name in ("C1", "C2", "C3", "C4"):
                if name == args.workload:
                    continue
                try:
                    result["per_config"][name] = time_config(torch, kcs, dev, name, 10 if name != "C4" else 10, 3)
                except Exception as e:
                    result["per_config"][name] = {"error": repr(e)}
            try:  # the launch-bound C1 (S:7-H6) as a batch of 100 noise realisations
                result["per_config"]["C1 x 100 replicas"] = time_replicas(torch, kcs, dev, "C1", 100, 10, 3)
            except Exception as e:
                result["per_config"]["C1 x 100 replicas"] = {"error": repr(e)}
        if not args.no_sweeps:
            try:
                result["sweeps"] = run_sweeps(torch, kcs, dev, peaks)
            except Exception as e:
                result["sweeps"] = {"error": repr(e)}
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(result), flush=True)


def run_e2e(ctx, cfg, prob, state0, torch, args, world, dist, dev):
    """kcs_icm_run_host with pinned host buffers: H2D (y, r, x, theta, lambda) and D2H (x, theta, lambda) every step."""
    x0, th0, lam0 = state0
    pin = lambda a: torch.tensor(np.asarray(a), dtype=torch.float32).contiguous().pin_memory()
    hy, hr = pin(prob["y"]), pin(prob["r"])
    hx, hth, hlam = pin(x0), pin(th0), pin(lam0)
    hx0, hth0 = torch.tensor(x0, dtype=torch.float32), torch.tensor(th0, dtype=torch.float32)
    scale, n_icm = float(prob["scale"]), cfg["n_icm"]
    big = input_bytes(cfg) > L2_BYTES
    flush = None if big else torch.empty(96 * 1024 * 1024, dtype=torch.float32, device=dev)

    def one(i):
        if i % n_icm == 0:
            hx.copy_(hx0); hth.copy_(hth0); hlam.zero_()
        if flush is not None:
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
def oracle_sample(cfg: dict, workload: str, for_baseline: bool):
    """A bounded sample of the workload for the oracle: the first nz_s slices (slices are independent direct planes
    in the OS pass and the LM cost is per voxel), with counts scaled by nz_s / nz.  cpu_baseline: 10-30 s of CPU
    work; --impl reference: every step a sample, sized so K + W steps end within a few minutes."""
    nz_s = ({"C1": 1, "C2": 8, "C3": 8, "C4": 3} if for_baseline else {"C1": 1, "C2": 2, "C3": 2, "C4": 1}).get(workload, 1)
    nz_s = min(nz_s, cfg["nz"])
    sub = dict(cfg, nz=nz_s, counts=cfg["counts"] * nz_s / cfg["nz"])  # 3-D phantoms: the central nz_s slices
    return sub, nz_s


def oracle_problem(workload: str, for_baseline: bool):
    from oracle import Oracle
    cfg = ki.config(workload)
    sub, nz_s = oracle_sample(cfg, workload, for_baseline)
    o = Oracle(sub)
    mask = o.default_mask()
    prob = ki.make_problem(sub, mask, o.kinetic_eval, o.forward_project, noisy=True)
    st = ki.initial_state(sub, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    return cfg, sub, nz_s, o, prob, st


def cpu_baseline(cfg: dict, workload: str) -> dict:
    """The oracle as it stands, one ICM iteration (beta = 0, the first of a reconstruction) on the bounded sample."""
    from oracle import Oracle
    _, sub, nz_s, o, prob, (x0, th0, lam0) = oracle_problem(workload, True)
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
    cfg, sub, nz_s, o, prob, (x0, th0, lam0) = oracle_problem(args.workload, False)
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
def run_sweeps(torch, kcs, dev, peaks) -> dict:
    """BASELINE configs[4] (C5) on the C4 geometry.  Inputs are made on the device (noiseless activity from the C4
    phantom) -- throughput only.  Every point carries its roofline fraction (SURVEY.md 8(d) max rule, bench.bounds)."""
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

    # (a) projector pair alone, frames batched per launch nf in {1, 4, 12, 29}; inputs (1.7 GB + 1.3 GB) exceed L2.
    # Stand-alone calls project the defined operation (no FOV clipping, all voxels).
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
        pt = {"frames_per_launch": nf, "launches": len(chunks),
              "forward_ms": ms_f, "forward_gsamples_s": sf / ms_f * 1e-6, "forward_kernel_ms": pf["forward"][0] / 2,
              "back_ms": ms_b, "back_gsamples_s": sf / ms_b * 1e-6, "back_kernel_ms": pb["back"][0] / 2}
        if peaks and "error" not in peaks:
            # all launches of the sweep point together: T frames in total whatever nf is
            wm = work_model(cfg, mask, T=T, subset=False, clipped=False)
            if nf < T:  # x (forward) / q (back) is re-read from HBM by every launch of nf frames only once: same bytes
                pass
            fb, bb = bounds(wm["forward"], pt["forward_kernel_ms"], peaks), bounds(wm["back"], pt["back_kernel_ms"], peaks)
            pt["forward_roofline"] = {"bound": fb["bound"], "frac": fb["frac"], "t_lb_ms": fb["t_lb_ms"], "l2_gbs": fb["l2_gbs"], "tflops": fb["tflops"]}
            pt["back_roofline"] = {"bound": bb["bound"], "frac": bb["frac"], "t_lb_ms": bb["t_lb_ms"], "l2_gbs": bb["l2_gbs"], "tflops": bb["tflops"]}
        out["projector"].append(pt)
    ctx.profile_enable(False)
    # (b) MAP-LM alone, 20 steps, start within +/-50 % of the truth, gamma in {0, 0.05, 0.5}
    rng = torch.Generator(device=dev)
    rng.manual_seed(4)
    start = (th_true * (0.5 + torch.rand(th_true.shape, generator=rng, device=dev))).contiguous()
    nfit = float(mask.sum()) * nz
    out["map_lm"] = []
    for gamma in (0.0, 0.05, 0.5):
        th_w = start.clone(); lam_w = torch.zeros((nz, ny, nx), dtype=torch.float32, device=dev)
        ctx.map_lm(x, th_w, lam_w, gamma, cfg["delta"], 20)  # warm-up
        torch.cuda.synchronize()
        th = start.clone(); lam = torch.zeros_like(lam_w)
        e0.record(); ctx.map_lm(x, th, lam, gamma, cfg["delta"], 20); e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        pt = {"gamma": gamma, "steps": 20, "ms": ms, "fits_s": nfit / ms * 1e3, "voxel_steps_s": nfit * 20 / ms * 1e3}
        if peaks and "error" not in peaks:
            flops = nfit * (21 * lm_flops_per_eval(T) + 20 * 500.0)  # 20 steps = 21 evaluations (the first step has two)
            pt["tflops"] = flops / ms * 1e-9
            pt["frac_of_fp32_peak"] = pt["tflops"] / peaks["fp32_tflops"]
            pt["frac_of_fp64_peak"] = pt["tflops"] / peaks["fp64_tflops"]
        out["map_lm"].append(pt)
    ctx.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C3", "C4"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweeps", action="store_true")
    ap.add_argument("--no-per-config", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
