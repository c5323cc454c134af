"""Pins for the oracle's OSL update, MAP-LM and ICM iteration (pins table)."""
import itertools

import numpy as np
import pytest

import kcs_inputs as ki
from oracle import Oracle


@pytest.fixture(scope="module")
def tiny():
    cfg = ki.small_config(nx=16, ny=16, n_angles=12, n_bins=16, n_subsets=3)
    o = Oracle(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    return cfg, o, mask, prob


def test_beta0_is_textbook_osem(tiny):
    """beta = 0  =>  x <- x / (A_s^T 1) * A_s^T (y / (A_s x + r))  (eq. 2 without the prior)."""
    cfg, o, mask, p = tiny
    x0, _, _ = ki.initial_state(cfg, mask, p["y"], p["r"], p["scale"], o.forward_project)
    F = np.ones_like(x0)
    x = o.os_pass(p["y"], p["r"], p["scale"], x0, F, beta=0.0)
    ref = x0.copy()
    S, A = cfg["n_subsets"], cfg["n_angles"]
    for s in range(S):
        yh = p["scale"] * o.forward_project(ref, s) + p["r"][:, None, None, None]
        q = p["y"][:, :, s::S, :] / yh
        bp = o.back_project(q, s)
        sens = o.sensitivity(s)
        with np.errstate(divide="ignore", invalid="ignore"):
            ref = np.where((mask > 0) & (sens > 1e-12 * sens.max()), ref * bp / sens, 0.0)
    np.testing.assert_allclose(x, ref, rtol=1e-12, atol=1e-300)
    assert np.all(x[:, :, mask == 0] == 0)


def test_prior_vanishes_when_F_equals_x(tiny):
    cfg, o, mask, p = tiny
    x0, _, _ = ki.initial_state(cfg, mask, p["y"], p["r"], p["scale"], o.forward_project)
    rng = np.random.default_rng(5)
    bp = rng.random(x0.shape)
    sens = o.sensitivity(0) * p["scale"]
    a = o.osl_update(x0, bp, sens, F=x0, beta=0.7)
    b = o.osl_update(x0, bp, sens, F=x0 * 3 + 1, beta=0.0)
    np.testing.assert_array_equal(a, b)


def test_prior_pulls_towards_F(tiny):
    """Q7: x above the model curve is pushed down, below is pushed up, relative to beta = 0; Q9 clamp."""
    cfg, o, mask, p = tiny
    x0 = np.ones((cfg["n_frames"], 1, 16, 16)) * mask
    sens = o.sensitivity(1)
    bp = np.broadcast_to(sens, x0.shape).copy()  # b = S -> beta=0 leaves x unchanged
    base = o.osl_update(x0, bp, sens, F=x0, beta=0.0)
    np.testing.assert_allclose(base[:, :, mask > 0], 1.0, rtol=1e-14)
    hi = o.osl_update(x0, bp, sens, F=0.5 * np.ones_like(x0), beta=0.1)  # x > F
    lo = o.osl_update(x0, bp, sens, F=2.0 * np.ones_like(x0), beta=0.1)  # x < F
    m = mask > 0
    assert np.all(hi[:, 0][:, m] < 1.0) and np.all(lo[:, 0][:, m] > 1.0)
    np.testing.assert_allclose(hi[:, 0][:, m], 1.0 / (1 + 0.1 * (1 - 0.5) / 0.5), rtol=1e-14)
    np.testing.assert_allclose(lo[:, 0][:, m], 1.0 / (1 + 0.1 * (1 - 2.0) / 2.0), rtol=1e-14)
    # Q9: denominator clamped at 0.1 S
    cl = o.osl_update(x0, bp, sens, F=1e3 * np.ones_like(x0), beta=5.0)
    np.testing.assert_allclose(cl[:, 0][:, m], 10.0, rtol=1e-14)
    # absolute mode: D = S + beta (x-F)/sigma2
    ab = o.osl_update(x0, bp, sens, F=0.5 * np.ones_like(x0), beta=0.2, prior_mode=1, sigma2=4.0)
    ref = sens[m] / (sens[m] + 0.2 * 0.5 / 4.0)
    np.testing.assert_allclose(ab[0, 0][m], ref, rtol=1e-13)


def test_consistent_data_is_fixed_point(tiny):
    """y = scale A x + r (noiseless, consistent)  =>  q = 1, b = S, x unchanged."""
    cfg, o, mask, p = tiny
    x = p["x_true"]
    out = o.os_pass(p["ybar"], p["r"], p["scale"], x, F=x, beta=0.3)
    np.testing.assert_allclose(out, x, rtol=1e-12, atol=1e-13)


def test_em_monotone_loglik_single_subset():
    """Q21: S = 1, beta = 0: Poisson log-likelihood is non-decreasing (EM theorem)."""
    cfg = ki.small_config(nx=16, ny=16, n_angles=12, n_bins=16, n_subsets=1)
    o = Oracle(cfg)
    mask = o.default_mask()
    p = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x, _, _ = ki.initial_state(cfg, mask, p["y"], p["r"], p["scale"], o.forward_project)
    ll = [o.poisson_loglik(p["y"], p["r"], p["scale"], x)]
    for _ in range(8):
        x = o.os_pass(p["y"], p["r"], p["scale"], x, F=x, beta=0.0)
        ll.append(o.poisson_loglik(p["y"], p["r"], p["scale"], x))
    d = np.diff(ll)
    assert np.all(d >= -1e-9 * abs(ll[0])), d
    assert ll[-1] > ll[0]


# ---------------------------------------------------------------------------------------------- MAP-LM

def test_noiseless_fixed_point():
    """x = F(xi_true), gamma = 0, start +/-50 %  =>  xi_true to 1e-6 (BASELINE north_star)."""
    cfg = ki.small_config(nx=8, ny=8, n_angles=8, n_bins=8, n_subsets=1, sched="C3")
    o = Oracle(cfg)
    mask = o.default_mask()
    _, th = ki.phantom(cfg)
    th = th * mask[None, None]
    x = o.kinetic_eval(th)
    start = ki.lm_start(th, seed=11)
    est, lam = o.map_lm(x, start, np.zeros((1, 8, 8)), gamma=0.0, delta=0.01, n_steps=60)
    m = mask > 0
    rel = np.abs(est[:, 0][:, m] - th[:, 0][:, m]) / np.abs(th[:, 0][:, m])
    assert rel.max() <= 1e-6, rel.max()
    # out-of-mask voxels untouched
    np.testing.assert_array_equal(est[:, 0][:, ~m], start[:, 0][:, ~m])


def test_cost_nonincreasing_and_jacobi_order():
    cfg = ki.small_config(nx=8, ny=8, n_angles=8, n_bins=8, n_subsets=1)
    o = Oracle(cfg)
    mask = o.default_mask()
    _, th = ki.phantom(cfg)
    th = th * mask[None, None]
    rng = np.random.default_rng(4)
    x = o.kinetic_eval(th) * (1 + 0.2 * rng.standard_normal((cfg["n_frames"], 1, 8, 8)))
    cur, lam = ki.lm_start(th, seed=12), np.zeros((1, 8, 8))
    gamma, delta = 1e5, 0.01
    # n_steps at once == one step at a time (state carried in theta, lambda only)
    a_th, a_lam = o.map_lm(x, cur, lam, gamma, delta, 3)
    b_th, b_lam = cur, lam
    for _ in range(3):
        b_th, b_lam = o.map_lm(x, b_th, b_lam, gamma, delta, 1)
    np.testing.assert_array_equal(a_th, b_th)
    np.testing.assert_array_equal(a_lam, b_lam)
    # Phi_v with neighbours frozen at the step's start never increases within a step (beyond the 1e-6 slack of Q15a)
    prev_th, prev_lam = cur, lam
    for _ in range(4):
        new_th, new_lam, cost = o.map_lm(x, prev_th, prev_lam, gamma, delta, 1, want_cost=True)
        for (j, i) in [(3, 3), (4, 2), (1, 4), (6, 5)]:
            nb = [prev_th[:, 0, j + dj, i + di] for dj, di in ((0, -1), (0, 1), (-1, 0), (1, 0))
                  if mask[j + dj, i + di]]
            before = o.lm_objective(x[:, 0, j, i], prev_th[:, 0, j, i], nb, gamma, delta)
            after = o.lm_objective(x[:, 0, j, i], new_th[:, 0, j, i], nb, gamma, delta)
            assert after <= before * (1 + 1e-6)
            assert abs(after - cost[0, j, i]) <= 1e-12 * max(1.0, abs(after))
        prev_th, prev_lam = new_th, new_lam


def test_huber_potential_through_objective():
    """H odd-symmetric derivative, |H'| <= delta, quadratic inside / linear outside (Q12)."""
    cfg = ki.small_config(nx=8, ny=8, n_angles=8, n_bins=8, n_subsets=1)
    o = Oracle(cfg)
    xi = np.array(ki.GREY)
    xv = o.kinetic_eval(xi.reshape(4, 1))[:, 0]  # zero data term
    delta, gamma = 0.01, 2.0

    def H(t):
        nb = xi.copy()
        nb[0] -= t  # xi_0 - nbr_0 = t, other parameters equal
        return o.lm_objective(xv, xi, [nb], gamma, delta) / gamma

    for t in (0.003, 0.01, 0.02, 0.5):
        ref = 0.5 * t * t if t <= delta else delta * t - 0.5 * delta * delta
        assert abs(H(t) - ref) < 1e-15 and abs(H(-t) - ref) < 1e-15
    slope = (H(0.5) - H(0.4)) / 0.1
    assert abs(slope - delta) < 1e-12


def test_large_gamma_pulls_to_neighbour_value():
    cfg = ki.small_config(nx=8, ny=8, n_angles=8, n_bins=8, n_subsets=1)
    o = Oracle(cfg)
    mask = o.default_mask()
    th = np.array(ki.WHITE)[:, None, None, None] * np.ones((4, 1, 8, 8)) * mask
    x = o.kinetic_eval(np.array(ki.GREY)[:, None, None, None] * np.ones((4, 1, 8, 8)) * mask)
    # delta huge => quadratic prior; gamma huge => each voxel stays at its (constant) neighbours' value
    est, _ = o.map_lm(x, th, np.zeros((1, 8, 8)), gamma=1e14, delta=10.0, n_steps=30)
    m = mask > 0
    np.testing.assert_allclose(est[:, 0][:, m], th[:, 0][:, m], rtol=1e-5)
    free, _ = o.map_lm(x, th, np.zeros((1, 8, 8)), gamma=0.0, delta=10.0, n_steps=30)
    np.testing.assert_allclose(free[:, 0][:, m], np.array(ki.GREY)[:, None] * np.ones(m.sum()), rtol=1e-5)


def test_brute_force_grid_optimum_8x8():
    """BASELINE north_star: brute-force grid search of the LM optimum on an 8x8 image.  Per voxel, Phi_v with
    frozen neighbours is minimised by nested 4-D grid refinement; LM's converged xi must reach the same minimum."""
    cfg = ki.small_config(nx=8, ny=8, n_angles=8, n_bins=8, n_subsets=1)
    o = Oracle(cfg)
    mask = o.default_mask()
    _, th = ki.phantom(cfg)
    th = th * mask[None, None]
    rng = np.random.default_rng(21)
    x = o.kinetic_eval(th) * (1 + 0.05 * rng.standard_normal((cfg["n_frames"], 1, 8, 8)))
    gamma, delta = 3e4, 0.01  # Q14: large enough for the prior to move the optimum
    frozen = th * (1 + 0.1 * rng.standard_normal(th.shape)) * mask[None, None]
    lo = np.array([0.0, 1e-4, 0.0, 0.0])
    hi = np.array([2.0, 2.0, 1.0, 1.0])
    for (j, i) in [(3, 4), (2, 2), (5, 3)]:
        nb = [frozen[:, 0, j + dj, i + di] for dj, di in ((0, -1), (0, 1), (-1, 0), (1, 0)) if mask[j + dj, i + di]]
        xv = x[:, 0, j, i]
        # (1) brute force: nested 5^4 grid refinement of Phi_v around the frozen value
        best = frozen[:, 0, j, i].copy()
        span = np.array([0.2, 0.3, 0.15, 0.1])
        phi_best = o.lm_objective(xv, best, nb, gamma, delta)
        for level in range(14):
            grids = [np.clip(best[p] + span[p] * np.linspace(-1, 1, 5), lo[p], hi[p]) for p in range(4)]
            for cand in itertools.product(*grids):
                ph = o.lm_objective(xv, np.array(cand), nb, gamma, delta)
                if ph < phi_best:
                    phi_best, best = ph, np.array(cand)
            span *= 0.5
        # (2) LM: one Jacobi step at a time, every other voxel reset to its frozen value after each step
        vol = frozen.copy()
        lam = np.zeros((1, 8, 8))
        cur = vol.copy()
        for _ in range(60):
            new, lam = o.map_lm(x, cur, lam, gamma, delta, 1)
            cur = vol.copy()
            cur[:, 0, j, i] = new[:, 0, j, i]  # keep every other voxel frozen
        phi_lm = o.lm_objective(xv, cur[:, 0, j, i], nb, gamma, delta)
        assert phi_lm <= phi_best * (1 + 1e-6), (phi_lm, phi_best)
        assert abs(phi_lm - phi_best) <= 2e-4 * abs(phi_best)
        # and the minimiser itself agrees where the objective is well conditioned (Ki = K1 k3/(k2+k3), vB)
        ki_lm = cur[0, 0, j, i] * cur[2, 0, j, i] / (cur[1, 0, j, i] + cur[2, 0, j, i])
        ki_bf = best[0] * best[2] / (best[1] + best[2])
        assert abs(ki_lm - ki_bf) <= 2e-2 * abs(ki_bf)


# ---------------------------------------------------------------------------------------------- ICM

def test_icm_iteration_is_the_composition(tiny):
    """I: F <- K(theta_old); OS pass with F fixed; theta <- MAP-LM(x_new).  beta=gamma=0 is OSEM + independent fits
    (PAPER.md:158 'INDIRECT'), gamma=0 is 'DIRECT'."""
    cfg, o, mask, p = tiny
    x0, th0, lam0 = ki.initial_state(cfg, mask, p["y"], p["r"], p["scale"], o.forward_project)
    for beta, gamma in ((0.0, 0.0), (0.1, 0.0), (0.1, 1e4)):
        x1, th1, lam1 = o.icm_iteration(p["y"], p["r"], p["scale"], x0, th0, lam0, beta, gamma, 0.01, 3)
        F = o.kinetic_eval(th0)
        xr = o.os_pass(p["y"], p["r"], p["scale"], x0, F, beta)
        thr, lamr = o.map_lm(xr, th0, lam0, gamma, 0.01, 3)
        np.testing.assert_array_equal(x1, xr)
        np.testing.assert_array_equal(th1, thr)
        np.testing.assert_array_equal(lam1, lamr)
    # r given as a full sinogram equals r given per frame
    rfull = np.broadcast_to(p["r"][:, None, None, None], p["y"].shape).copy()
    xa = o.os_pass(p["y"], rfull, p["scale"], x0, x0, 0.0)
    xb = o.os_pass(p["y"], p["r"], p["scale"], x0, x0, 0.0)
    np.testing.assert_array_equal(xa, xb)


def test_icm_runs_and_improves(tiny):
    """Sanity on the frozen readings (SURVEY.md 8(c) 'End-to-end sanity'): finite, log-likelihood rises,
    activity error falls over a few ICM iterations on Poisson data."""
    cfg, o, mask, p = tiny
    x, th, lam = ki.initial_state(cfg, mask, p["y"], p["r"], p["scale"], o.forward_project)
    ll = [o.poisson_loglik(p["y"], p["r"], p["scale"], x)]
    err = [np.linalg.norm(x - p["x_true"]) / np.linalg.norm(p["x_true"])]
    for it in range(4):
        x, th, lam = o.icm_iteration(p["y"], p["r"], p["scale"], x, th, lam, 0.0 if it == 0 else 0.1, 0.05, 0.01, 5)
        assert np.all(np.isfinite(x)) and np.all(np.isfinite(th))
        ll.append(o.poisson_loglik(p["y"], p["r"], p["scale"], x))
        err.append(np.linalg.norm(x - p["x_true"]) / np.linalg.norm(p["x_true"]))
    assert ll[-1] > ll[0] and err[-1] < err[0]
    assert np.all(th[:, :, mask == 0] == 0) and np.all(x[:, :, mask == 0] == 0)


def test_icm_joint_fixed_point_and_contraction(tiny):
    """I on CONSISTENT data, y = scale A x* + r with x* = K(theta*): the pair (x*, theta*) is a fixed point of
    the whole iteration with the kinetic prior on -- the ratio is 1, the prior term vanishes at x = F, the fit's gradient
    vanishes at x = K(theta) -- and from a perturbed theta the iteration moves back towards it.  With uniform maps the
    Huber gradient vanishes too (in-mask neighbours only), so the fixed point survives gamma > 0."""
    cfg, o, mask, p = tiny
    m = mask > 0
    lam0 = np.zeros((cfg["nz"], cfg["ny"], cfg["nx"]))
    th, xs = p["theta_true"], p["x_true"]
    x1, th1, _ = o.icm_iteration(p["ybar"], p["r"], p["scale"], xs, th, lam0, 0.1, 0.0, 0.01, 3)
    assert np.abs(x1 - xs).max() <= 1e-10 * xs.max()
    assert np.abs(th1 - th).max() <= 1e-8
    # perturbed maps, exact activity: one iteration (5 LM steps) removes most of the perturbation, the prior's pull on x
    # (towards the curve of the perturbed maps) stays a fraction of the distance between the two curves
    th_p = th * (1.0 + 0.1 * (ki.uniform(th.shape, seed=5) - 0.5))
    F_p = o.kinetic_eval(th_p) * mask[None, None]
    x2, th2, _ = o.icm_iteration(p["ybar"], p["r"], p["scale"], xs, th_p, lam0, 0.1, 0.0, 0.01, 5)
    e0 = np.linalg.norm((th_p - th)[:, :, m])
    e2 = np.linalg.norm((th2 - th)[:, :, m])
    assert e2 < 0.5 * e0, (e0, e2)
    assert np.linalg.norm(x2 - xs) < 0.5 * np.linalg.norm(F_p - xs)
    assert np.linalg.norm(x2 - xs) > 0  # beta = 0.1 did act
    # uniform maps, Huber prior on
    th_u = np.array(ki.THETA0)[:, None, None, None] * mask[None, None].astype(np.float64)
    x_u = o.kinetic_eval(th_u) * mask[None, None]
    y_u = p["scale"] * o.forward_project(x_u, -1) + p["r"][:, None, None, None]
    x3, th3, _ = o.icm_iteration(y_u, p["r"], p["scale"], x_u, th_u, lam0, 0.1, 1e4, 0.01, 3)
    assert np.abs(x3 - x_u).max() <= 1e-10 * x_u.max()
    assert np.abs(th3 - th_u)[:, :, m].max() <= 1e-8
