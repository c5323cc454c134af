"""Oracle against itself: how far does the 10-iteration ICM chain amplify an fp32-sized perturbation of the activity?

BASELINE.json north_star asks, after 10 ICM iterations, for every kinetic parameter within 1e-3 on >= 99.9 % of the
voxels.  One OS pass of ANY fp32 implementation leaves x with a relative error of a few 1e-7 (S subsets x ~8 roundings of
6e-8 each: measured 2.7e-7 rel-L2 for the CUDA path on C2, tests/test_gpu_fullsize.py).  This experiment runs the fp64
oracle twice on the same data -- chain A untouched, chain B with x multiplied by (1 + 2.7e-7 N(0,1)) after the OS pass of
every iteration, nothing else changed -- and counts the voxels of B that leave the 1e-3 band around A.  The oracle's
arithmetic is not involved in the comparison (both chains are the oracle): the loss is a property of the ITERATION
(noise-dominated 4-parameter fits with parameters on their bounds move by > 1e-3 under a 3e-7 change of the curve they
fit), i.e. the floor under which no fp32 OS pass can stay.  Measured with KCS_FLOOR_FULL=1 (C2 at full size, 8 slices):
min over the parameters 99.82 % after 10 iterations (profiles/r2_oracle_noise_floor_C2.txt); the CUDA path reaches
99.85-99.88 % on the same data.  KCS_FLOOR_FULL=C3 (C3 at full size, 2 counts per voxel-frame): 98.93 %, activity 1.26e-3
(profiles/r2_oracle_noise_floor_C3.txt); the CUDA path: 98.8 %, 1.30e-3.  KCS_FLOOR_FULL=C4z4 (C4's in-plane geometry on 4
slices, the third chain of tests/test_gpu_fullsize.py): 98.98 %, 1.79e-3 (profiles/r2_oracle_noise_floor_C4z4.txt); the CUDA
path: 98.7 %, 2.2e-3.  The default run uses 2 slices of C2 so that the CPU suite stays short.

    KCS_FLOOR_FULL=1 python -m pytest tests/test_oracle_noise_floor.py -s -q
"""
import os

import numpy as np

import kcs_inputs as ki
from oracle import Oracle

FLOORS = np.array([0.05, 0.05, 0.02, 0.02])  # Q19
RMS = 2.7e-7


def chain_pair(cfg, rms, seed=99):
    f32 = lambda a: np.float32(a).astype(np.float64)
    o = Oracle(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    x0, th0, r, scale = f32(x0), f32(th0), f32(prob["r"]), float(np.float32(prob["scale"]))
    m3 = np.broadcast_to(mask[None] > 0, th0.shape[1:])
    rng = np.random.Generator(np.random.PCG64(seed))
    A = B = (x0, th0, lam0)
    rows = []
    for it in range(cfg["n_icm"]):
        beta = 0.0 if it == 0 else cfg["beta"]
        A = o.icm_iteration(prob["y"], r, scale, *A, beta, cfg["gamma"], cfg["delta"], cfg["n_lm"])
        xb, thb, lamb = o.icm_iteration(prob["y"], r, scale, *B, beta, cfg["gamma"], cfg["delta"], 0)  # OS pass only
        xb = xb * (1.0 + rms * rng.standard_normal(xb.shape))
        thb, lamb = o.map_lm(xb, thb, lamb, cfg["gamma"], cfg["delta"], cfg["n_lm"])
        B = (xb, thb, lamb)
        ok = np.abs(B[1] - A[1]) <= 1e-3 * np.maximum(np.abs(A[1]), FLOORS[:, None, None, None])
        rows.append((float(np.linalg.norm(B[0] - A[0]) / np.linalg.norm(A[0])), [float(ok[p][m3].mean()) for p in range(4)]))
    return rows


def test_fp32_sized_perturbation_is_amplified_past_the_tolerance_band():
    env = os.environ.get("KCS_FLOOR_FULL", "")
    full = env in ("1", "C2", "C3", "C4z4")
    name = env if env in ("C3", "C4z4") else "C2"    # KCS_FLOOR_FULL=C3: the same experiment on C3 at full size (~10 min)
    if name == "C4z4":                               # C4's in-plane geometry on 4 slices, the chain of tests/test_gpu_fullsize.py
        cfg = (lambda c: dict(c, nz=4, counts=c["counts"] * 4 / c["nz"]))(ki.config("C4"))
    else:
        cfg = ki.config(name)
    if not full:
        cfg = dict(cfg, nz=2, counts=cfg["counts"] * 2 / cfg["nz"])
    rows = chain_pair(cfg, RMS)
    for it, (ex, fr) in enumerate(rows):
        print(f"{name}{'' if full else ' (2 slices)'} rms {RMS:g} iteration {it + 1}: activity rel-L2 {ex:.3e} "
              f"parameter fractions within 1e-3 {['%.5f' % a for a in fr]}")
    ex1, fr1 = rows[0]
    ex10, fr10 = rows[-1]
    assert 0.5 * RMS <= ex1 <= 2.0 * RMS and min(fr1) >= 0.9999      # one iteration: the perturbation itself, no loss
    assert ex10 >= 30.0 * RMS                                       # ten iterations: amplified by orders of magnitude
    assert min(fr10) < 0.9997                                       # and voxels have left the band ...
    assert min(fr10) > 0.97                                         # ... a per cent of them at most
    if full:
        assert min(fr10) < 0.999                                    # at full size: below BASELINE's 99.9 %
