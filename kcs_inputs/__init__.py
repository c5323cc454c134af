"""Seeded synthetic inputs for the KCS hot path -- shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no projector, no kinetic model, no LM): it
only describes the workloads of BASELINE.json (geometry, frame schedules, phantom label maps and
region parameters, random draws).  Where a workload needs model values (noise-free sinograms, the
initial image), the caller passes in the functions that compute them -- the oracle's in the oracle
tests, the CUDA library's in bench.py -- so no value ever flows from one implementation to the other.

They stand in for the paper's simulated phantom and its Siemens mMR FDG brain
scan, neither of which is available; the recipes are BASELINE.json `configs`
with the readings Q2, Q6, Q17, Q18, Q20 of SURVEY.md section 8(c) (repeated in DESIGN.md).
"""
from __future__ import annotations

import numpy as np

FENG_A = (851.1, 21.88, 20.81)
FENG_LAMBDA = (4.134, 0.1191, 0.01043)

# (K1, k2, k3, vB) -- BASELINE.json configs[0] item (4)
GREY = (0.102, 0.130, 0.062, 0.05)
WHITE = (0.054, 0.109, 0.045, 0.03)
BACKGROUND = (0.03, 0.10, 0.01, 0.02)
ZERO_UPTAKE = (0.0, 0.10, 0.0, 0.0)

THETA0 = (0.05, 0.10, 0.03, 0.03)  # Q17 initial maps


def _frames(spec):
    d = np.concatenate([np.full(n, float(sec)) for n, sec in spec]) / 60.0
    e = np.concatenate([[0.0], np.cumsum(d)])
    return e[:-1].copy(), e[1:].copy()


_SCHED = {
    "C1": [(4, 30), (4, 120), (4, 300)],
    "C2": [(8, 15), (4, 60), (4, 120), (8, 240)],
    "C3": [(12, 10), (6, 30), (5, 60), (6, 300)],
}


def config(name: str) -> dict:
    """Geometry / schedule / hyper-parameters of workload C1..C5 (C5 = C4 geometry)."""
    name = name.upper()
    base = dict(feng_A=FENG_A, feng_lambda=FENG_LAMBDA, beta=0.1, gamma=0.05, delta=0.01, n_lm=5, n_icm=10)
    if name == "C1":
        ts, te = _frames(_SCHED["C1"])
        base.update(name="C1", nx=64, ny=64, nz=1, vx=2.0, vy=2.0, vz=2.0, n_angles=60, n_bins=64, bin_mm=2.0,
                    n_steps=64, step_mm=2.0, n_subsets=4, counts=2e6, seed=0)
    elif name == "C2":
        ts, te = _frames(_SCHED["C2"])
        base.update(name="C2", nx=128, ny=128, nz=8, vx=2.0, vy=2.0, vz=2.0, n_angles=120, n_bins=128, bin_mm=2.0,
                    n_steps=128, step_mm=2.0, n_subsets=6, counts=8e6 * 8, seed=1)
    elif name == "C3":
        ts, te = _frames(_SCHED["C3"])
        base.update(name="C3", nx=128, ny=128, nz=64, vx=2.0, vy=2.0, vz=2.0, n_angles=168, n_bins=128, bin_mm=2.0,
                    n_steps=128, step_mm=2.0, n_subsets=21, counts=5e7, seed=2)
    elif name in ("C4", "C5"):
        ts, te = _frames(_SCHED["C3"])
        base.update(name=name, nx=344, ny=344, nz=127, vx=2.09, vy=2.09, vz=2.03, n_angles=252, n_bins=344,
                    bin_mm=2.09, n_steps=344, step_mm=2.09, n_subsets=21, counts=2e8, seed=3 if name == "C4" else 4)
    else:
        raise ValueError(name)
    base["t_start_min"], base["t_end_min"] = ts, te
    base["n_frames"] = len(ts)
    return base


def small_config(nx=16, ny=16, nz=1, n_angles=12, n_bins=16, n_subsets=3, sched="C1", **kw) -> dict:
    """A tiny config for unit tests (same conventions; K = nx steps of one voxel)."""
    ts, te = _frames(_SCHED[sched])
    c = dict(name="tiny", feng_A=FENG_A, feng_lambda=FENG_LAMBDA, beta=0.1, gamma=0.05, delta=0.01, n_lm=5,
             n_icm=10, nx=nx, ny=ny, nz=nz, vx=2.0, vy=2.0, vz=2.0, n_angles=n_angles, n_bins=n_bins, bin_mm=2.0,
             n_steps=nx, step_mm=2.0, n_subsets=n_subsets, counts=3e5, seed=7,
             t_start_min=ts, t_end_min=te, n_frames=len(ts))
    c.update(kw)
    return c


def _grid(cfg):
    X = (np.arange(cfg["nx"]) - 0.5 * (cfg["nx"] - 1)) * cfg["vx"]
    Y = (np.arange(cfg["ny"]) - 0.5 * (cfg["ny"] - 1)) * cfg["vy"]
    Z = (np.arange(cfg["nz"]) - 0.5 * (cfg["nz"] - 1)) * cfg["vz"]
    return np.meshgrid(Z, Y, X, indexing="ij")


def _ell(Z, Y, X, c, ax):
    zz = ((Z - c[2]) / ax[2]) ** 2 if ax[2] > 0 else 0.0
    return ((X - c[0]) / ax[0]) ** 2 + ((Y - c[1]) / ax[1]) ** 2 + zz <= 1.0


def phantom(cfg: dict):
    """Label map [nz,ny,nx] (0 background, 1 white, 2 grey, 3 zero-uptake, 4 lesion) and theta_true[4,nz,ny,nx].

    Q20: head semi-axes (0.842 R, R); grey rim/shell = head minus the head shrunk by the rim thickness;
    random grey regions by rejection inside the white interior; PCG64(seed), draw order radius -> cx -> cy (-> cz).
    """
    name = cfg["name"]
    rng = np.random.Generator(np.random.PCG64(cfg["seed"]))
    Z, Y, X = _grid(cfg)
    nz = cfg["nz"]
    lab = np.zeros(Z.shape, dtype=np.int8)
    k1scale = np.ones(Z.shape)
    big = 1e30
    if name in ("C1", "C2", "tiny"):
        R = {"C1": 55.0, "C2": 110.0}.get(name, 0.40 * cfg["ny"] * cfg["vy"])
        rim = 6.0 if name != "tiny" else 0.2 * R
        ax = (0.842 * R, R, big)
        head = _ell(Z, Y, X, (0, 0, 0), ax)
        inner = _ell(Z, Y, X, (0, 0, 0), (ax[0] - rim, ax[1] - rim, big))
        lab[head] = 2
        lab[inner] = 1
        ndisk = {"C1": 3, "C2": 6}.get(name, 2)
        rlo, rhi = (4.0, 8.0) if name != "tiny" else (0.1 * R, 0.2 * R)
        for z in range(nz):
            placed = 0
            while placed < ndisk:
                r = rng.uniform(rlo, rhi)
                cx = rng.uniform(-ax[0], ax[0])
                cy = rng.uniform(-ax[1], ax[1])
                # rejection: the disk must lie inside the white interior
                if ((abs(cx) + r) / (ax[0] - rim)) ** 2 + ((abs(cy) + r) / (ax[1] - rim)) ** 2 > 1.0:
                    continue
                d = (X[z] - cx) ** 2 + (Y[z] - cy) ** 2 <= r * r
                lab[z][d] = 2
                placed += 1
    elif name == "C3":
        ax = (0.842 * 110.0, 110.0, 58.0)
        shell = 6.0
        head = _ell(Z, Y, X, (0, 0, 0), ax)
        inner = _ell(Z, Y, X, (0, 0, 0), tuple(a - shell for a in ax))
        lab[head] = 2
        lab[inner] = 1
        placed = 0
        while placed < 10:
            sa = rng.uniform(5.0, 15.0, size=3)
            c = rng.uniform(-1, 1, size=3) * np.array(ax)
            if sum(((abs(c[i]) + sa[i]) / (ax[i] - shell)) ** 2 for i in range(3)) > 1.0:
                continue
            lab[_ell(Z, Y, X, c, sa)] = 2
            placed += 1
    elif name in ("C4", "C5"):
        ax = (80.0, 95.0, 65.0)
        shell = 3.0
        head = _ell(Z, Y, X, (0, 0, 0), ax)
        inner = _ell(Z, Y, X, (0, 0, 0), tuple(a - shell for a in ax))
        lab[head] = 2
        lab[inner] = 1
        for sx in (-1.0, 1.0):  # basal ganglia (grey) and ventricles (zero uptake)
            lab[_ell(Z, Y, X, (sx * 18.0, 5.0, 0.0), (8.0, 14.0, 10.0))] = 2
            lab[_ell(Z, Y, X, (sx * 7.0, -8.0, 10.0), (4.5, 18.0, 8.0))] = 3
        placed = 0
        while placed < 20:
            r = rng.uniform(3.0, 10.0)
            c = rng.uniform(-1, 1, size=3) * np.array(ax)
            if sum(((abs(c[i]) + r) / (ax[i] - shell)) ** 2 for i in range(3)) > 1.0:
                continue
            m = _ell(Z, Y, X, c, (r, r, r)) & (lab != 3)
            lab[m] = 4
            k1scale[m] = 1.5
            placed += 1
    else:
        raise ValueError(name)
    table = np.array([BACKGROUND, WHITE, GREY, ZERO_UPTAKE, GREY], dtype=np.float64)
    theta = np.moveaxis(table[lab], -1, 0).copy()
    theta[0] *= k1scale
    return lab, theta


def poisson(mean: np.ndarray, seed: int) -> np.ndarray:
    """Q20: Poisson noise from PCG64(seed + 1000)."""
    rng = np.random.Generator(np.random.PCG64(seed + 1000))
    return rng.poisson(np.maximum(mean, 0.0)).astype(np.float64)


def noise_realisations(ybar: np.ndarray, seed: int, n: int) -> np.ndarray:
    """P:131 ("100 noisy realizations"): n independent Poisson draws of one noise-free sinogram ybar[T,nz,A,B], stacked
    replica-major along z -> [T, n*nz, A, B].  Realisation k uses PCG64(seed + 1000 + k), so realisation 0 is `poisson`."""
    return np.concatenate([poisson(ybar, seed + k) for k in range(n)], axis=1)


def tile_replicas(a: np.ndarray, axis: int, n: int) -> np.ndarray:
    """The same array for every replica, replica-major along the slice axis."""
    return np.concatenate([a] * n, axis=axis)


MU_WATER_511KEV = 0.0096  # 1/mm, linear attenuation coefficient of water / soft tissue at 511 keV


def attenuation_factors(cfg: dict, forward_project) -> np.ndarray:
    """SURVEY 8(f)3 stand-in for a measured attenuation map: the head of the phantom (every labelled tissue) is
    water, n[z,a,b] = exp(-mu * chord length) with the chord lengths from the caller's forward projector applied to the
    head's indicator image (mm).  Returns [nz, A, B] in (0, 1]."""
    lab, _ = phantom(cfg)
    head = (lab > 0).astype(np.float64)
    chord = np.asarray(forward_project(head[None]), dtype=np.float64)[0]
    return np.exp(-MU_WATER_511KEV * chord)


def lm_start(theta_true: np.ndarray, seed: int) -> np.ndarray:
    """C5(b): initial parameters uniform within +/-50 % of the truth."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return theta_true * rng.uniform(0.5, 1.5, size=theta_true.shape)


def uniform(shape, seed: int, lo=0.0, hi=1.0) -> np.ndarray:
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.uniform(lo, hi, size=shape)


def make_problem(cfg: dict, mask: np.ndarray, kinetic_eval, forward_project, noisy: bool = True) -> dict:
    """Assemble one workload.  `kinetic_eval(theta[4,nz,ny,nx]) -> F[T,nz,ny,nx]` and
    `forward_project(x[T,nz,ny,nx]) -> ybar[T,nz,A,B]` (all angles, no scale) are supplied by the caller.

    Q6: scale = N_true / sum(A x_true); r_t = 0.1 * mean_d(scale * A x_true,t); y ~ Poisson(scale A x + r).
    """
    lab, theta_true = phantom(cfg)
    theta_true = theta_true * mask[None, None].astype(np.float64)
    x_true = np.asarray(kinetic_eval(theta_true), dtype=np.float64) * mask[None, None]
    proj = np.asarray(forward_project(x_true), dtype=np.float64)
    scale = float(cfg["counts"]) / float(proj.sum())
    T = proj.shape[0]
    r = 0.1 * scale * proj.reshape(T, -1).mean(axis=1)
    ybar = scale * proj + r[:, None, None, None]
    y = poisson(ybar, cfg["seed"]) if noisy else ybar
    return dict(labels=lab, theta_true=theta_true, x_true=x_true, scale=scale, r=r, ybar=ybar, y=y)


def initial_state(cfg: dict, mask: np.ndarray, y: np.ndarray, r: np.ndarray, scale: float, forward_project):
    """Q17: x0_t = per-frame constant matching the frame's net counts inside the mask; theta0 constant in the
    mask; lambda = 0 (uninitialised)."""
    T = y.shape[0]
    nz, ny, nx = cfg["nz"], cfg["ny"], cfg["nx"]
    m3 = np.broadcast_to(mask[None].astype(np.float64), (nz, ny, nx)).copy()
    pm = float(np.asarray(forward_project(m3[None]), dtype=np.float64).sum())
    net = np.maximum(y.reshape(T, -1).sum(axis=1) - r * y[0].size, 1e-3 * y.reshape(T, -1).sum(axis=1) + 1e-12)
    x0 = (net / (scale * pm))[:, None, None, None] * m3[None]
    theta0 = np.array(THETA0)[:, None, None, None] * m3[None]
    lam0 = np.zeros((nz, ny, nx))
    return x0, theta0, lam0
