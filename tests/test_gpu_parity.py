"""GPU parity: every C-ABI call of include/kcs.h against the fp64 oracle on the same seeded inputs.

Tolerances are BASELINE.json north_star's: per-call relative L2 <= 1e-5 (projection, back-projection),
<= 1e-4 (one OSL update); after 10 ICM iterations activity relative L2 <= 1e-3 and each kinetic parameter within
1e-3 relative (Q19 floors) on >= 99.9 % of in-mask voxels.
"""
import numpy as np
import pytest

import kcs_inputs as ki
from oracle import Oracle

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

FLOORS = np.array([0.05, 0.05, 0.02, 0.02])  # Q19


def _kcs():
    import paper_1803_10045_b200 as kcs
    return kcs


def dev(a):
    return torch.tensor(np.asarray(a), dtype=torch.float32, device="cuda").contiguous()


def host(t):
    return t.detach().cpu().numpy().astype(np.float64)


def rel_l2(g, o):
    return float(np.linalg.norm((g - o).ravel()) / max(np.linalg.norm(o.ravel()), 1e-300))


def close(g, o, tol):
    """BJ's tolerance is a relative L2; a whole-array norm hides a wrong edge bin or border voxel, so every parity check
    also bounds the largest element-wise error: max|g - o| <= tol max|o|."""
    g, o = np.asarray(g), np.asarray(o)
    return rel_l2(g, o) <= tol and float(np.abs(g - o).max()) <= tol * float(np.abs(o).max())


def param_ok_fraction(thg, tho, mask):
    ok = np.abs(thg - tho) <= 1e-3 * np.maximum(np.abs(tho), FLOORS[:, None, None, None])
    return [float(ok[p][:, mask > 0].mean()) for p in range(4)]


CONFIGS = {
    "tiny": lambda: ki.small_config(nx=16, ny=16, nz=1, n_angles=12, n_bins=16, n_subsets=3),
    # ragged: odd sizes, non-square, bins != nx, K != nx, T = 12 -> several tiles with tails in every kernel
    "ragged": lambda: ki.small_config(nx=45, ny=37, nz=3, n_angles=30, n_bins=51, n_subsets=5, n_steps=57),
    "C1": lambda: ki.config("C1"),
    "C2": lambda: ki.config("C2"),
    # anisotropic voxels / finer bins (C4-like ratios on a small grid), T = 29
    "aniso": lambda: ki.small_config(nx=40, ny=48, nz=2, n_angles=36, n_bins=64, n_subsets=4, sched="C3",
                                     vx=2.0, vy=2.2, bin_mm=2.1, step_mm=2.15, n_steps=60),
}


@pytest.fixture(scope="module", params=["tiny", "ragged", "C1", "aniso"])
def pair(request):
    cfg = CONFIGS[request.param]()
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    yield cfg, o, ctx
    ctx.close()


def test_mask_matches(pair):
    cfg, o, ctx = pair
    assert np.array_equal(ctx.mask(), o.default_mask())


@pytest.mark.parametrize("subset", [-1, 0, 2])
def test_forward_project(pair, subset):
    cfg, o, ctx = pair
    T = cfg["n_frames"]
    x = ki.uniform((T, cfg["nz"], cfg["ny"], cfg["nx"]), seed=11, lo=0.0, hi=2.0)
    x32 = np.float32(x).astype(np.float64)
    yo = o.forward_project(x32, subset)
    y = torch.zeros(yo.shape, dtype=torch.float32, device="cuda")
    ctx.forward_project(dev(x32), y, subset)
    assert close(host(y), yo, 1e-5)
    # per-frame too (a frame must not leak into its neighbour)
    for f in (0, T - 1):
        assert close(host(y)[f], yo[f], 1e-5)


@pytest.mark.parametrize("subset", [-1, 1])
def test_back_project(pair, subset):
    cfg, o, ctx = pair
    T = cfg["n_frames"]
    As = o.n_sub_angles(subset)
    q = np.float32(ki.uniform((T, cfg["nz"], As, cfg["n_bins"]), seed=12, lo=0.0, hi=2.0)).astype(np.float64)
    bo = o.back_project(q, subset)
    b = torch.zeros(bo.shape, dtype=torch.float32, device="cuda")
    ctx.back_project(dev(q), b, subset)
    assert close(host(b), bo, 1e-5)
    assert close(host(b)[T - 1], bo[T - 1], 1e-5)


def test_frame_ranges(pair):
    """C5(a): frames batched nf at a time must reproduce the all-frames result exactly (same arithmetic per frame)."""
    cfg, o, ctx = pair
    T = cfg["n_frames"]
    x = dev(ki.uniform((T, cfg["nz"], cfg["ny"], cfg["nx"]), seed=13))
    y_all = torch.zeros((T, cfg["nz"], cfg["n_angles"], cfg["n_bins"]), dtype=torch.float32, device="cuda")
    ctx.forward_project(x, y_all)
    y_part = torch.full_like(y_all, -7.0)
    for f0, nf in ((0, 1), (1, 4), (5, T - 5)):
        ctx.forward_project(x, y_part, -1, f0, nf)
    assert torch.equal(y_all, y_part)
    b_all = torch.zeros_like(x)
    ctx.back_project(y_all, b_all)
    b_part = torch.full_like(x, -7.0)
    for f0, nf in ((0, 3), (3, 1), (4, T - 4)):
        ctx.back_project(y_all, b_part, -1, f0, nf)
    assert torch.equal(b_all, b_part)


def test_no_cross_slice_or_border_leak(pair):
    """Slices are independent direct planes and the padded borders must stay zero: with the neighbouring slices (and
    frames) filled with 1e20 an out-of-slice tap or a clipped ray that reads past its slice shows up in the result."""
    cfg, o, ctx = pair
    T, nz = cfg["n_frames"], cfg["nz"]
    if nz < 3:
        pytest.skip("needs three slices")
    x = np.float32(ki.uniform((T, nz, cfg["ny"], cfg["nx"]), seed=61, lo=0.0, hi=2.0)).astype(np.float64)
    xb = x.copy()
    xb[:, 0] *= 1e20
    xb[:, 2] *= 1e20
    y = torch.zeros((T, nz, cfg["n_angles"], cfg["n_bins"]), dtype=torch.float32, device="cuda")
    ctx.forward_project(dev(xb), y)
    yo = o.forward_project(x, -1)
    assert close(host(y)[:, 1], yo[:, 1], 1e-5)
    q = np.float32(ki.uniform(yo.shape, seed=62, lo=0.0, hi=2.0)).astype(np.float64)
    qb = q.copy()
    qb[:, 0] *= 1e20
    qb[:, 2] *= 1e20
    b = torch.zeros((T, nz, cfg["ny"], cfg["nx"]), dtype=torch.float32, device="cuda")
    ctx.back_project(dev(qb), b)
    bo = o.back_project(q, -1)
    assert close(host(b)[:, 1], bo[:, 1], 1e-5)
    # and a later ordinary call is unaffected by what the previous one left in the workspace
    ctx.forward_project(dev(x), y)
    assert close(host(y), yo, 1e-5)


def test_bitwise_repeatable(pair):
    """No atomics anywhere on the path (BJ north_star): two runs from the same state agree bit for bit."""
    cfg, o, ctx = pair
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    y, r = dev(prob["y"]), dev(prob["r"])
    outs = []
    for _ in range(2):
        x, th, lam = dev(x0), dev(th0), dev(lam0)
        ctx.icm_iteration(y, r, float(prob["scale"]), x, th, lam, 0.0, cfg["gamma"], cfg["delta"], 2)
        ctx.icm_iteration(y, r, float(prob["scale"]), x, th, lam, 0.1, cfg["gamma"], cfg["delta"], 2)
        outs.append((x.clone(), th.clone(), lam.clone()))
    for a, b in zip(*outs):
        assert torch.equal(a, b)


def test_adjointness_gpu(pair):
    cfg, o, ctx = pair
    T = cfg["n_frames"]
    x = dev(ki.uniform((T, cfg["nz"], cfg["ny"], cfg["nx"]), seed=14))
    q = dev(ki.uniform((T, cfg["nz"], cfg["n_angles"], cfg["n_bins"]), seed=15))
    y = torch.zeros_like(q)
    b = torch.zeros_like(x)
    ctx.forward_project(x, y)
    ctx.back_project(q, b)
    lhs = float((y.double() * q.double()).sum())
    rhs = float((x.double() * b.double()).sum())
    assert abs(lhs - rhs) <= 2e-6 * abs(lhs)


def test_sensitivity(pair):
    cfg, o, ctx = pair
    for s in (-1, 0, cfg["n_subsets"] - 1):
        sg = torch.zeros((cfg["ny"], cfg["nx"]), dtype=torch.float32, device="cuda")
        ctx.sensitivity(s, sg)
        assert close(host(sg), o.sensitivity(s), 1e-5)


@pytest.mark.parametrize("mode", [0, 1])
def test_osl_update(pair, mode):
    cfg, o, ctx = pair
    T = cfg["n_frames"]
    shp = (T, cfg["nz"], cfg["ny"], cfg["nx"])
    f = lambda a: np.float32(a).astype(np.float64)
    x = f(ki.uniform(shp, 21, 0.5, 5.0))
    bp = f(ki.uniform(shp, 22, 0.0, 3.0))
    F = f(ki.uniform(shp, 23, 0.2, 6.0))
    sens = f(o.sensitivity(1) * 0.37)
    xo = o.osl_update(x, bp, sens, F, 0.1, mode, 2.5)
    xg = dev(x)
    ctx.osl_update(xg, dev(bp), dev(sens), dev(F), 0.1, mode, 2.5)
    assert close(host(xg), xo, 1e-5)
    m = ctx.mask()
    assert np.all(host(xg)[:, :, m == 0] == 0)


def test_one_os_pass_through_icm(pair):
    """One OSL pass (n_lm = 0): fused ratio + back-projection + OSL over all subsets, <= 1e-4."""
    cfg, o, ctx = pair
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    th0 = np.float32(th0).astype(np.float64)
    x0 = np.float32(x0).astype(np.float64)
    for beta in (0.0, 0.1):
        xo, tho, _ = o.icm_iteration(prob["y"], np.float32(prob["r"]).astype(np.float64), float(np.float32(prob["scale"])),
                                     x0, th0, lam0, beta, 0.0, 0.01, 0)
        x, th, lam = dev(x0), dev(th0), dev(lam0)
        ctx.icm_iteration(dev(prob["y"]), dev(prob["r"]), float(prob["scale"]), x, th, lam, beta, 0.0, 0.01, 0)
        assert close(host(x), xo, 1e-4)
        assert np.array_equal(host(th), tho)
        # full randoms sinogram gives the same result as the per-frame constant
        rfull = np.broadcast_to(np.float32(prob["r"])[:, None, None, None], prob["y"].shape)
        x2, th2, lam2 = dev(x0), dev(th0), dev(lam0)
        ctx.icm_iteration(dev(prob["y"]), dev(rfull), float(prob["scale"]), x2, th2, lam2, beta, 0.0, 0.01, 0)
        assert torch.equal(x, x2)


def _theta_box(n, seed):
    """Parameters over the whole box incl. the physiological range and a = k2+k3 hugging lambda_2, lambda_3 and 0."""
    rng = np.random.Generator(np.random.PCG64(seed))
    th = np.empty((4, n))
    th[0] = rng.uniform(0.0, 2.0, n)
    th[1] = rng.uniform(1e-4, 2.0, n)
    th[2] = rng.uniform(0.0, 1.0, n)
    th[3] = rng.uniform(0.0, 1.0, n)
    q = n // 4
    th[0, :q] = rng.uniform(0.01, 0.2, q)
    th[1, :q] = rng.uniform(0.05, 0.2, q)
    th[2, :q] = rng.uniform(0.0, 0.1, q)
    th[3, :q] = rng.uniform(0.0, 0.1, q)
    k = 0
    for lam in ki.FENG_LAMBDA[1:]:
        for d in (0.0, 1e-7, -1e-7, 1e-5, -1e-5, 9e-5, -9e-5, 1.1e-4, -1.1e-4, 1e-3, -1e-3):
            a = lam + d
            k3 = min(0.3 * a, 0.5 * a)
            th[1, q + k] = a - k3
            th[2, q + k] = k3
            k += 1
    for a in (1e-4, 2e-4, 1e-3, 1e-2):  # tiny a: k2 at / near its lower bound, k3 = 0 or tiny
        th[1, q + k] = a
        th[2, q + k] = 0.0
        k += 1
        th[1, q + k] = 1e-4
        th[2, q + k] = a
        k += 1
    return th


@pytest.mark.parametrize("sched", ["C1", "C2", "C3"])
def test_kinetic_eval_over_parameter_box(sched):
    """H1: max relative error of F_m <= 5e-6 over the whole box (fp32 storage of theta and F included)."""
    nx, ny, nz = 64, 32, 2
    cfg = ki.small_config(nx=nx, ny=ny, nz=nz, n_angles=8, n_bins=64, n_subsets=2, sched=sched)
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    T = cfg["n_frames"]
    th = np.float32(_theta_box(nx * ny * nz, 31)).astype(np.float64).reshape(4, nz, ny, nx)
    Fo, Jo = o.kinetic_eval(th, jac=True)
    F = torch.zeros((T, nz, ny, nx), dtype=torch.float32, device="cuda")
    J = torch.zeros((4, T, nz, ny, nx), dtype=torch.float32, device="cuda")
    ctx.kinetic_eval(dev(th), F, J)
    Fg, Jg = host(F), host(J)
    assert np.max(np.abs(Fg - Fo) / np.maximum(np.abs(Fo), 1e-3)) <= 5e-6
    scaleJ = np.max(np.abs(Jo), axis=1, keepdims=True)
    assert np.max(np.abs(Jg - Jo) / np.maximum(scaleJ, 1e-3)) <= 5e-6
    F2 = torch.zeros_like(F)
    ctx.kinetic_eval(dev(th), F2, None)
    assert torch.equal(F, F2)
    ctx.close()


def _lm_problem(cfg, o, seed, noise):
    mask = o.default_mask()
    _, th_true = ki.phantom(cfg)
    th_true = th_true * mask[None, None]
    x = o.kinetic_eval(th_true) * mask[None, None]
    rng = np.random.Generator(np.random.PCG64(seed))
    x = x * (1.0 + noise * rng.standard_normal(x.shape))
    start = ki.lm_start(th_true, seed + 1)
    return mask, np.float32(x).astype(np.float64), np.float32(start).astype(np.float64), th_true


@pytest.mark.parametrize("gamma,delta,noise", [(0.0, 0.01, 0.0), (0.05, 0.01, 0.1), (3e5, 0.01, 0.1), (2e6, 0.05, 0.3)])
def test_map_lm(pair, gamma, delta, noise):
    """L1-L3: n synchronised steps; lambda carried; Huber prior at gamma values where it bites (Q14, H7)."""
    cfg, o, ctx = pair
    mask, x, start, th_true = _lm_problem(cfg, o, 41, noise)
    lam0 = np.zeros(x.shape[1:])
    for n_steps in (1, 4):
        tho, lamo, costo = o.map_lm(x, start, lam0, gamma, delta, n_steps, want_cost=True)
        th, lam = dev(start), dev(lam0)
        cost = torch.zeros(x.shape[1:], dtype=torch.float32, device="cuda")
        ctx.map_lm(dev(x), th, lam, gamma, delta, n_steps, cost)
        fr = param_ok_fraction(host(th), tho, mask)
        assert min(fr) >= 0.999, (n_steps, fr)
        m = mask > 0
        lg, cg = host(lam)[:, m], host(cost)[:, m]
        assert np.mean(np.abs(lg - lamo[:, m]) <= 1e-3 * np.abs(lamo[:, m])) >= 0.999
        assert np.mean(np.abs(cg - costo[:, m]) <= 1e-3 * np.abs(costo[:, m]) + 1e-6) >= 0.999
        assert np.array_equal(host(th)[:, :, ~m], start[:, :, ~m])  # out-of-mask voxels untouched


@pytest.mark.parametrize("gamma", [0.0, 0.05, 0.5])
def test_map_lm_c5b_recipe(gamma):
    """BASELINE configs[4](b) on a small volume: 20 LM steps, start uniform within +/-50 % of the truth, gamma swept over
    0, 0.05, 0.5 (noisy curves, three slices so that the z-neighbours take part)."""
    cfg = ki.small_config(nx=40, ny=40, nz=3, n_angles=8, n_bins=40, n_subsets=2, sched="C3")
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    mask, x, start, th_true = _lm_problem(cfg, o, 47, 0.15)
    lam0 = np.zeros(x.shape[1:])
    tho, lamo, costo = o.map_lm(x, start, lam0, gamma, 0.01, 20, want_cost=True)
    th, lam = dev(start), dev(lam0)
    cost = torch.zeros(x.shape[1:], dtype=torch.float32, device="cuda")
    ctx.map_lm(dev(x), th, lam, gamma, 0.01, 20, cost)
    fr = param_ok_fraction(host(th), tho, mask)
    assert min(fr) >= 0.999, fr
    m = mask > 0
    assert np.mean(np.abs(host(cost)[:, m] - costo[:, m]) <= 1e-3 * np.abs(costo[:, m]) + 1e-6) >= 0.999
    ctx.close()


def test_map_lm_noiseless_recovers_truth():
    cfg = ki.config("C1")
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    mask, x, start, th_true = _lm_problem(cfg, o, 43, 0.0)
    th, lam = dev(start), dev(np.zeros(x.shape[1:]))
    ctx.map_lm(dev(x), th, lam, 0.0, 0.01, 40, None)
    thg = host(th)
    m = mask > 0
    err = np.abs(thg - th_true)[:, :, m] / np.maximum(np.abs(th_true[:, :, m]), FLOORS[:, None, None])
    assert np.quantile(err, 0.999) <= 2e-4  # fp32 storage of x and theta limits this (not 1e-6 as in fp64)
    ctx.close()


@pytest.mark.parametrize("name", ["C1", "ragged"])
def test_icm_10_iterations(name):
    """BJ north_star: after 10 ICM iterations activity rel-L2 <= 1e-3, parameters within 1e-3 on >= 99.9 % of voxels."""
    cfg = CONFIGS[name]()
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    f = lambda a: np.float32(a).astype(np.float64)
    x0, th0, r, scale = f(x0), f(th0), f(prob["r"]), float(np.float32(prob["scale"]))
    xo, tho, lamo = x0, th0, lam0
    for it in range(cfg["n_icm"]):
        beta = 0.0 if it == 0 else cfg["beta"]
        xo, tho, lamo = o.icm_iteration(prob["y"], r, scale, xo, tho, lamo, beta, cfg["gamma"], cfg["delta"], cfg["n_lm"])
    y, rd = dev(prob["y"]), dev(r)
    x, th, lam = dev(x0), dev(th0), dev(lam0)
    for it in range(cfg["n_icm"]):
        beta = 0.0 if it == 0 else cfg["beta"]
        ctx.icm_iteration(y, rd, scale, x, th, lam, beta, cfg["gamma"], cfg["delta"], cfg["n_lm"])
    ex = rel_l2(host(x), xo)
    fr = param_ok_fraction(host(th), tho, mask)
    print(name, "activity rel-L2", ex, "param fractions", fr)
    assert ex <= 1e-3
    assert min(fr) >= 0.999, fr
    # kcs_icm_run (y packed once) and the host-buffer entry give the same iterates as 10 single calls
    x2, th2, lam2 = dev(x0), dev(th0), dev(lam0)
    ctx.icm_run(y, rd, scale, x2, th2, lam2, 0.0, cfg["beta"], cfg["gamma"], cfg["delta"], cfg["n_lm"], cfg["n_icm"])
    assert torch.equal(x2, x) and torch.equal(th2, th) and torch.equal(lam2, lam)  # bit for bit: same kernels, same order
    hx, hth, hlam = np.float32(x0), np.float32(th0), np.float32(lam0)
    ctx.icm_run_host(np.float32(prob["y"]), np.float32(r), scale, hx, hth, hlam, 0.0, cfg["beta"], cfg["gamma"],
                     cfg["delta"], cfg["n_lm"], cfg["n_icm"])
    assert np.array_equal(hx, x2.cpu().numpy())
    assert np.array_equal(hth, th2.cpu().numpy())
    ctx.close()


def test_host_entry_moves_the_volume_in_z_chunks():
    """kcs_icm_run_host copies x and y in z chunks (>= 16 slices each) while earlier chunks go through their OS pass, and
    returns x chunk by chunk; direct planes are independent, so the result must equal kcs_icm_run bit for bit -- for one
    iteration (copy-in and copy-out chunked in the same pass) and for three."""
    # 96 x 96 x 64, T = 29: the whole volume is past the forward projector's K-split threshold (148 x 2048 ray lanes), one
    # of its four 16-slice chunks alone is not -- the split must be decided on the whole volume
    cfg = ki.small_config(nx=96, ny=96, nz=64, n_angles=24, n_bins=96, n_subsets=3, counts=4e6, sched="C3")
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    y, rd, scale = dev(prob["y"]), dev(prob["r"]), float(prob["scale"])
    for n_iter in (1, 3):
        x, th, lam = dev(x0), dev(th0), dev(lam0)
        ctx.icm_run(y, rd, scale, x, th, lam, 0.0, cfg["beta"], cfg["gamma"], cfg["delta"], 2, n_iter)
        hx, hth, hlam = np.float32(x0), np.float32(th0), np.float32(lam0)
        ctx.icm_run_host(np.float32(prob["y"]), np.float32(prob["r"]), scale, hx, hth, hlam, 0.0, cfg["beta"], cfg["gamma"],
                         cfg["delta"], 2, n_iter)
        assert np.array_equal(hx, x.cpu().numpy()) and np.array_equal(hth, th.cpu().numpy())
        assert np.array_equal(hlam, lam.cpu().numpy())
    # full randoms sinogram and pinned buffers take the same path
    rfull = np.ascontiguousarray(np.broadcast_to(np.float32(prob["r"])[:, None, None, None], prob["y"].shape))
    px = torch.tensor(np.float32(x0)).pin_memory(); pth = torch.tensor(np.float32(th0)).pin_memory()
    plam = torch.tensor(np.float32(lam0)).pin_memory()
    ctx.icm_run_host(torch.tensor(np.float32(prob["y"])).pin_memory(), torch.tensor(rfull).pin_memory(), scale, px, pth, plam,
                     0.0, cfg["beta"], cfg["gamma"], cfg["delta"], 2, 3)
    assert np.array_equal(px.numpy(), hx) and np.array_equal(pth.numpy(), hth)
    ctx.close()


def test_host_entry_lead_chunk_and_two_lanes():
    """With slices as large as C4's (344 x 344, 252 x 344, T = 29) the host pipeline starts with a short lead chunk (4
    slices), doubles the chunk size from there (8, then the remaining 20 of 32) and runs alternate chunks on two
    streams: still kcs_icm_run bit for bit.  Inputs: seeded noise, no oracle needed for an equality."""
    cfg = dict(ki.config("C4"), nz=32)
    ctx = _kcs().Context(cfg)
    T, nz, ny, nx, A, B = cfg["n_frames"], 32, cfg["ny"], cfg["nx"], cfg["n_angles"], cfg["n_bins"]
    mask = ctx.mask()
    y0 = np.float32(np.floor(4.0 * ki.uniform((T, nz, A, B), seed=61)))
    r0 = np.float32(0.05 + 0.01 * np.arange(T))
    x0 = np.float32((0.5 + ki.uniform((T, nz, ny, nx), seed=62)) * mask)
    th0 = np.float32(np.broadcast_to(np.array([0.1, 0.1, 0.05, 0.05])[:, None, None, None], (4, nz, ny, nx))
                     * (0.8 + 0.4 * ki.uniform((4, nz, ny, nx), seed=63)))
    lam0 = np.zeros((nz, ny, nx), dtype=np.float32)
    for n_iter in (1, 2):
        x, th, lam = dev(x0), dev(th0), dev(lam0)
        ctx.icm_run(dev(y0), dev(r0), 1.0, x, th, lam, 0.0, cfg["beta"], cfg["gamma"], cfg["delta"], 2, n_iter)
        hx, hth, hlam = x0.copy(), th0.copy(), lam0.copy()
        ctx.icm_run_host(y0, r0, 1.0, hx, hth, hlam, 0.0, cfg["beta"], cfg["gamma"], cfg["delta"], 2, n_iter)
        assert np.isfinite(hx).all() and float(np.abs(hx).max()) > 0
        assert np.array_equal(hx, x.cpu().numpy()) and np.array_equal(hth, th.cpu().numpy())
        assert np.array_equal(hlam, lam.cpu().numpy())
    ctx.close()


def test_projector_C2_full_size():
    """C2 geometry (128x128x8, 120x128, T = 24): several blocks per slice and z-batching in the back-projector."""
    cfg = CONFIGS["C2"]()
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    T = cfg["n_frames"]
    x = np.float32(ki.uniform((T, cfg["nz"], cfg["ny"], cfg["nx"]), seed=51)).astype(np.float64)
    yo = o.forward_project(x, -1)
    y = torch.zeros(yo.shape, dtype=torch.float32, device="cuda")
    ctx.forward_project(dev(x), y)
    assert close(host(y), yo, 1e-5)
    q = np.float32(ki.uniform(yo.shape, seed=52)).astype(np.float64)
    bo = o.back_project(q, -1)
    b = torch.zeros(x.shape, dtype=torch.float32, device="cuda")
    ctx.back_project(dev(q), b)
    assert close(host(b), bo, 1e-5)
    ctx.close()


def test_user_stream_ordering():
    """Every call is enqueued on the stream given at create / kcs_set_stream and never synchronises: work issued on a
    side stream (inputs prepared there, the second-stream overlap inside kcs_icm_iteration included) gives bit for bit
    the default-stream result once that stream is synchronised."""
    kcs = _kcs()
    cfg = CONFIGS["ragged"]()
    o = Oracle(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    ref = kcs.Context(cfg)
    y, r = dev(prob["y"]), dev(prob["r"])
    xr, thr, lamr = dev(x0), dev(th0), dev(lam0)
    for beta in (0.0, 0.1):
        ref.icm_iteration(y, r, float(prob["scale"]), xr, thr, lamr, beta, cfg["gamma"], cfg["delta"], 3)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    ctx = kcs.Context(cfg, stream=side.cuda_stream)
    with torch.cuda.stream(side):
        xs, ths, lams = dev(x0), dev(th0), dev(lam0)       # produced on the side stream, consumed in order
        for beta in (0.0, 0.1):
            ctx.icm_iteration(y, r, float(prob["scale"]), xs, ths, lams, beta, cfg["gamma"], cfg["delta"], 3)
    side.synchronize()
    assert torch.equal(xs, xr) and torch.equal(ths, thr) and torch.equal(lams, lamr)
    # moving the context to another stream later works the same way
    other = torch.cuda.Stream()
    ctx.set_stream(other.cuda_stream)
    with torch.cuda.stream(other):
        x2, th2, lam2 = dev(x0), dev(th0), dev(lam0)
        for beta in (0.0, 0.1):
            ctx.icm_iteration(y, r, float(prob["scale"]), x2, th2, lam2, beta, cfg["gamma"], cfg["delta"], 3)
    other.synchronize()
    assert torch.equal(x2, xr) and torch.equal(th2, thr)
    ctx.close()
    ref.close()


def test_error_codes():
    kcs = _kcs()
    cfg = CONFIGS["tiny"]()
    bad = dict(cfg, n_subsets=5)
    with pytest.raises(kcs.KcsError) as e:
        kcs.Context(bad)
    assert e.value.code == -3
    ts, te = ki._frames([(40, 10)])
    with pytest.raises(kcs.KcsError) as e:
        kcs.Context(dict(cfg, t_start_min=ts, t_end_min=te, n_frames=40))
    assert e.value.code == -4
    with pytest.raises(kcs.KcsError) as e:
        kcs.Context(dict(cfg, bin_mm=0.5))
    assert e.value.code == -2
    ctx = kcs.Context(cfg)
    x = torch.zeros((cfg["n_frames"], 1, 16, 16), dtype=torch.float32, device="cuda")
    y = torch.zeros((cfg["n_frames"], 1, 4, 16), dtype=torch.float32, device="cuda")
    with pytest.raises(kcs.KcsError) as e:
        ctx._check(ctx._lib.kcs_forward_project(ctx._h, x.data_ptr(), y.data_ptr(), 7, 0, 1))
    assert e.value.code == -2
    with pytest.raises(kcs.KcsError) as e:
        ctx._check(ctx._lib.kcs_forward_project(ctx._h, None, y.data_ptr(), 0, 0, 1))
    assert e.value.code == -1
    ctx.close()
