"""INDIRECT / DIRECT / KCS-DIRECT on N noise realisations of one phantom.

The three methods of P:156-160 are parameter settings of the same ICM path:

    INDIRECT    beta = 0, gamma = 0: n_icm OS passes (plain OSEM of every frame), THEN the voxel-wise fit
                (n_icm * n_lm LM steps on the final images);
    DIRECT      beta > 0, gamma = 0: the ICM loop with the kinetic prior, no spatial prior on the maps;
    KCS         beta > 0, gamma > 0: the ICM loop with the kinetic prior and the Huber prior (the paper's method).

All N realisations are reconstructed in ONE batch: the context is created with n_replicas = N and every kernel launch
covers N * nz slices (kcs.h).  The macro-parameter map K_i = K1 k3 / (k2 + k3) comes from kcs_ki_map.  Only
argument marshalling and the final bias / variance bookkeeping (numpy, over the N maps) happen here; every step of the
reconstruction runs in libkcs.so.

    python -m paper_1803_10045_b200.methods --workload C1 --replicas 16
"""
from __future__ import annotations

import argparse
import json

import numpy as np

METHODS = ("INDIRECT", "DIRECT", "KCS")
REGIONS = {0: "background", 1: "white", 2: "grey", 4: "lesion"}


def reconstruct(ctx, method: str, y, r, scale: float, x0, th0, lam0, cfg: dict):
    """One method on the batched volume; tensors are float32 CUDA tensors in kcs.h layouts (replica-major).  Returns
    (x, theta, K_i) device tensors."""
    import torch
    x, th, lam = x0.clone(), th0.clone(), lam0.clone()
    n_icm, n_lm, beta, gamma, delta = cfg["n_icm"], cfg["n_lm"], cfg["beta"], cfg["gamma"], cfg["delta"]
    if method == "INDIRECT":
        ctx.icm_run(y, r, scale, x, th, lam, 0.0, 0.0, 0.0, delta, 0, n_icm)       # OSEM only
        ctx.map_lm(x, th, lam, 0.0, delta, n_icm * n_lm)                          # post-reconstruction fit
    elif method == "DIRECT":
        ctx.icm_run(y, r, scale, x, th, lam, 0.0, beta, 0.0, delta, n_lm, n_icm)
    elif method == "KCS":
        ctx.icm_run(y, r, scale, x, th, lam, 0.0, beta, gamma, delta, n_lm, n_icm)
    else:
        raise ValueError(method)
    ki = torch.zeros_like(lam)
    ctx.ki_map(th, ki)
    return x, th, ki


def region_stats(ki_maps: np.ndarray, labels: np.ndarray, ki_true: np.ndarray, mask: np.ndarray) -> dict:
    """per region, over the N realisations ki_maps[N, nz, ny, nx]: mean relative bias of the voxel means and
    mean coefficient of variation (std over realisations / truth), both in per cent."""
    mean, std = ki_maps.mean(axis=0), ki_maps.std(axis=0, ddof=1) if ki_maps.shape[0] > 1 else np.zeros(ki_maps.shape[1:])
    out = {}
    for lab, name in REGIONS.items():
        m = (labels == lab) & (mask[None] > 0) & (ki_true > 0)
        if not m.any():
            continue
        out[name] = {"voxels": int(m.sum()), "ki_true": float(ki_true[m].mean()),
                     "bias_pct": float(100.0 * ((mean[m] - ki_true[m]) / ki_true[m]).mean()),
                     "cov_pct": float(100.0 * (std[m] / ki_true[m]).mean())}
    return out


def run(workload: str = "C1", n_replicas: int = 8, gamma: float | None = None, device: str = "cuda") -> dict:
    """Build `n_replicas` Poisson realisations of the workload's phantom, reconstruct them with the three methods and
    return the per-region K_i statistics.  The noise-free data come from this library's own forward model."""
    import torch

    import kcs_inputs as ki
    from . import Context

    base = ki.config(workload)
    if gamma is not None:
        base = dict(base, gamma=gamma)
    cfg = dict(base, n_replicas=n_replicas)
    T, nz, ny, nx, A, B = base["n_frames"], base["nz"], base["ny"], base["nx"], base["n_angles"], base["n_bins"]
    dev = torch.device(device)
    one = Context(base)                      # a single-replica context makes the noise-free data and the start image
    f32 = lambda a: torch.tensor(np.asarray(a), dtype=torch.float32, device=dev).contiguous()

    def kin(theta):
        F = torch.zeros((T, nz, ny, nx), dtype=torch.float32, device=dev)
        one.kinetic_eval(f32(theta), F)
        return F.cpu().numpy().astype(np.float64)

    def fwd(x):
        x = np.asarray(x)
        xd = torch.zeros((T, nz, ny, nx), dtype=torch.float32, device=dev)
        xd[:x.shape[0]] = f32(x)
        yd = torch.zeros((T, nz, A, B), dtype=torch.float32, device=dev)
        one.forward_project(xd, yd, -1, 0, x.shape[0])
        return yd[:x.shape[0]].cpu().numpy().astype(np.float64)

    mask = one.mask()
    prob = ki.make_problem(base, mask, kin, fwd, noisy=False)
    x0, th0, lam0 = ki.initial_state(base, mask, prob["ybar"], prob["r"], prob["scale"], fwd)
    one.close()
    y = ki.noise_realisations(prob["ybar"], base["seed"], n_replicas)
    ctx = Context(cfg)
    yd, rd = f32(y), f32(prob["r"])
    x0d, th0d, lam0d = f32(ki.tile_replicas(x0, 1, n_replicas)), f32(ki.tile_replicas(th0, 1, n_replicas)), \
        f32(ki.tile_replicas(lam0, 0, n_replicas))
    th_true = prob["theta_true"]
    a = th_true[1] + th_true[2]
    ki_true = np.where(a > 0, th_true[0] * th_true[2] / np.where(a > 0, a, 1.0), 0.0)
    out = {"workload": workload, "n_replicas": n_replicas, "gamma": cfg["gamma"], "beta": cfg["beta"], "methods": {}}
    for m in METHODS:
        n0 = ctx.launch_count()
        _, _, kid = reconstruct(ctx, m, yd, rd, float(prob["scale"]), x0d, th0d, lam0d, cfg)
        torch.cuda.synchronize()
        kim = kid.cpu().numpy().astype(np.float64).reshape(n_replicas, nz, ny, nx)
        out["methods"][m] = {"regions": region_stats(kim, prob["labels"], ki_true, mask),
                             "gpu_launches": ctx.launch_count() - n0}
    ctx.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="C1", choices=["C1", "C2"])
    ap.add_argument("--replicas", type=int, default=8)
    ap.add_argument("--gamma", type=float, default=None, help="Huber weight of KCS (default: the workload's)")
    args = ap.parse_args()
    print(json.dumps(run(args.workload, args.replicas, args.gamma)))


if __name__ == "__main__":
    main()
