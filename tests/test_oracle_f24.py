"""Pins for the oracle's fit options: frame weights (weighted least squares), the 3x3-clique
neighbourhood of P:114 (8 in-plane neighbours + the two axial ones) and one Huber threshold per parameter map.  The
neighbour gathering, the weights and the thresholds are redone here with numpy indexing; special cases reduce to the
unweighted fit and to a shorter frame schedule."""
import numpy as np
import pytest

import kcs_inputs as ki
from oracle import Oracle


@pytest.fixture(autouse=True)
def _restore_defaults():
    yield
    Oracle.set_lm_options()


def _problem(nx=5, ny=6, nz=3, sched="C1", seed=3):
    cfg = ki.small_config(nx=nx, ny=ny, nz=nz, n_angles=8, n_bins=max(nx, ny), n_subsets=2, sched=sched)
    rng = np.random.default_rng(seed)
    shp = (nz, ny, nx)
    base = np.array(ki.GREY)[:, None, None, None]
    th_true = base * (1 + 0.3 * rng.uniform(-1, 1, size=(4,) + shp))
    start = base * (1 + 0.3 * rng.uniform(-1, 1, size=(4,) + shp))
    mask = np.ones((ny, nx), dtype=np.uint8)
    o = Oracle(cfg, mask=mask)
    x = o.kinetic_eval(th_true) * (1 + 0.05 * rng.standard_normal((cfg["n_frames"],) + shp))
    return cfg, o, mask, x, start


def _huber(t, d):
    a = np.abs(t)
    return np.where(a <= d, 0.5 * t * t, d * a - 0.5 * d * d)


def test_cost_with_weights_clique_neighbourhood_and_per_parameter_delta():
    """Phi_v returned by kcso_map_lm after one step = 1/2 sum_m w_m (x_m - F_m(theta_new))^2 + gamma sum_p sum_k
    H_{delta_p}(theta_new,p - theta_prev,k,p) over the 8 in-plane + 2 axial in-mask neighbours of the PREVIOUS iterate,
    recomputed here from the oracle's (separately pinned) model curve with numpy gathering."""
    cfg, o, mask, x, start = _problem()
    mask = mask.copy()
    mask[0, 0] = mask[5, 4] = mask[2, 3] = 0
    o = Oracle(cfg, mask=mask)
    T = cfg["n_frames"]
    w = np.linspace(0.2, 1.7, T)
    d4 = np.array([0.004, 0.02, 0.007, 0.011])
    gamma = 3e5
    Oracle.set_lm_options(frame_w=w, neighbourhood=10, delta4=d4)
    prev, lam = start * mask[None, None], np.zeros((3, 6, 5))
    offs = [(0, 0, -1), (0, 0, 1), (0, -1, 0), (0, 1, 0), (-1, 0, 0), (1, 0, 0), (0, -1, -1), (0, -1, 1), (0, 1, -1), (0, 1, 1)]
    for step in range(2):
        new, lam_new, cost = o.map_lm(x, prev, lam, gamma, 123.0, 1, want_cost=True)   # the scalar delta is ignored
        F = o.kinetic_eval(new)
        for z in range(3):
            for j in range(6):
                for i in range(5):
                    if not mask[j, i]:
                        assert cost[z, j, i] == 0.0
                        continue
                    phi = 0.5 * np.sum(w * (x[:, z, j, i] - F[:, z, j, i]) ** 2)
                    for dz, dj, di in offs:
                        zz, jj, ii = z + dz, j + dj, i + di
                        if 0 <= zz < 3 and 0 <= jj < 6 and 0 <= ii < 5 and mask[jj, ii]:
                            phi += gamma * np.sum(_huber(new[:, z, j, i] - prev[:, zz, jj, ii], d4))
                    assert abs(phi - cost[z, j, i]) <= 1e-10 * max(1.0, abs(phi)), (step, z, j, i)
        prev, lam = new, lam_new
    # not vacuous: the diagonal neighbours and the per-parameter thresholds change the result
    Oracle.set_lm_options(frame_w=w, neighbourhood=6, delta4=d4)
    six = o.map_lm(x, start * mask[None, None], np.zeros((3, 6, 5)), gamma, 123.0, 2)[0]
    assert np.abs(six - prev).max() > 1e-4
    Oracle.set_lm_options(frame_w=w, neighbourhood=10)
    one_delta = o.map_lm(x, start * mask[None, None], np.zeros((3, 6, 5)), gamma, 0.004, 2)[0]
    assert np.abs(one_delta - prev).max() > 1e-5


def test_unit_weights_are_the_plain_fit_and_a_common_factor_changes_nothing():
    cfg, o, mask, x, start = _problem()
    lam0 = np.zeros((3, 6, 5))
    plain = o.map_lm(x, start, lam0, 3e4, 0.01, 4, want_cost=True)
    Oracle.set_lm_options(frame_w=np.ones(cfg["n_frames"]), neighbourhood=6, delta4=[0.01] * 4)
    same = o.map_lm(x, start, lam0, 3e4, 0.5, 4, want_cost=True)
    for a, b in zip(plain, same):
        assert np.array_equal(a, b)
    # gamma = 0: Phi -> c Phi, J^T W J -> c J^T W J, lambda_0 = 1e-3 max diag -> c lambda_0: the steps do not change
    Oracle.set_lm_options(frame_w=np.full(cfg["n_frames"], 1.0))
    th1, lam1, c1 = o.map_lm(x, start, lam0, 0.0, 0.01, 5, want_cost=True)
    Oracle.set_lm_options(frame_w=np.full(cfg["n_frames"], 7.0))
    th7, lam7, c7 = o.map_lm(x, start, lam0, 0.0, 0.01, 5, want_cost=True)
    np.testing.assert_allclose(th7, th1, rtol=1e-10, atol=1e-13)
    np.testing.assert_allclose(lam7, 7.0 * lam1, rtol=1e-10)
    np.testing.assert_allclose(c7, 7.0 * c1, rtol=1e-10)


def test_zero_weight_drops_the_frame():
    """w_m = 0 on the last two frames is the fit of the first T - 2 frames: the same answer as a context whose schedule
    simply ends two frames earlier (frames are contiguous from t = 0, so the remaining frame integrals are the same)."""
    cfg, o, mask, x, start = _problem()
    T = cfg["n_frames"]
    w = np.ones(T)
    w[-2:] = 0.0
    lam0 = np.zeros((3, 6, 5))
    Oracle.set_lm_options(frame_w=w)
    th_w, lam_w, c_w = o.map_lm(x, start, lam0, 0.0, 0.01, 5, want_cost=True)
    Oracle.set_lm_options()
    short = dict(cfg, t_start_min=cfg["t_start_min"][:-2], t_end_min=cfg["t_end_min"][:-2], n_frames=T - 2)
    o2 = Oracle(short, mask=mask)
    th_s, lam_s, c_s = o2.map_lm(x[:-2], start, lam0, 0.0, 0.01, 5, want_cost=True)
    np.testing.assert_allclose(th_w, th_s, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(c_w, c_s, rtol=1e-12)


def test_curvature_with_no_data_is_one_newton_step_to_the_neighbour_mean():
    """All frame weights 0: Phi = gamma sum_p sum_k H(xi_p - xi_k,p), a quadratic while every difference is inside delta.
    With the Huber curvature in the LM matrix, lambda_0 = 1e-3 max diag J^T W J = 0 and M = gamma n_k I, so one step lands
    every voxel EXACTLY on the mean of its neighbours in the previous iterate -- a different code path from the
    gradient, checked here against numpy means.  (Without the curvature the matrix is zero and the step is rejected.)"""
    cfg, o, mask, x, start = _problem(nx=5, ny=4, nz=3)
    T = cfg["n_frames"]
    rng = np.random.default_rng(5)
    prev = np.array(ki.GREY)[:, None, None, None] * (1 + 0.01 * rng.uniform(-1, 1, size=(4, 3, 4, 5)))
    lam0 = np.zeros((3, 4, 5))
    Oracle.set_lm_options(frame_w=np.zeros(T), neighbourhood=10, delta4=[1.0] * 4, prior_curvature=True)
    new, lam, cost = o.map_lm(x, prev, lam0, 2.5, 0.0, 1, want_cost=True)
    offs = [(0, 0, -1), (0, 0, 1), (0, -1, 0), (0, 1, 0), (-1, 0, 0), (1, 0, 0), (0, -1, -1), (0, -1, 1), (0, 1, -1), (0, 1, 1)]
    for z in range(3):
        for j in range(4):
            for i in range(5):
                nb = [prev[:, z + dz, j + dj, i + di] for dz, dj, di in offs
                      if 0 <= z + dz < 3 and 0 <= j + dj < 4 and 0 <= i + di < 5]
                np.testing.assert_allclose(new[:, z, j, i], np.mean(nb, axis=0), rtol=1e-13)
    Oracle.set_lm_options(frame_w=np.zeros(T), neighbourhood=10, delta4=[1.0] * 4, prior_curvature=False)
    stuck = o.map_lm(x, prev, lam0, 2.5, 0.0, 1)[0]
    assert np.array_equal(stuck, prev)


def test_fixed_parameter_gives_the_one_tissue_model():
    """box k3 in [0, 0]: the fit of the one-tissue compartment model.  Noise-free one-tissue curves are recovered to 1e-6
    from a +-30 % start, k3 stays exactly 0 and takes no part in the solve; the default box is untouched by a reset."""
    cfg, o, mask, x, start = _problem(nx=4, ny=4, nz=1)
    rng = np.random.default_rng(9)
    th_true = np.array([0.08, 0.12, 0.0, 0.04])[:, None, None, None] * (1 + 0.2 * rng.uniform(-1, 1, size=(4, 1, 4, 4)))
    th_true[2] = 0.0
    x = o.kinetic_eval(th_true)
    start = th_true * (1 + 0.3 * rng.uniform(-1, 1, size=th_true.shape))
    start[2] = 0.05                                   # a wrong k3 in the start: the fixed value must replace it
    Oracle.set_lm_options(box_lo=[0.0, 1e-4, 0.0, 0.0], box_hi=[2.0, 2.0, 0.0, 1.0])
    th, lam = o.map_lm(x, start, np.zeros((1, 4, 4)), 0.0, 0.01, 60)
    assert np.all(th[2] == 0.0)
    np.testing.assert_allclose(th[[0, 1, 3]], th_true[[0, 1, 3]], rtol=1e-6)
    Oracle.set_lm_options()
    th2 = th_true.copy()
    th2[2] = 0.05
    free = o.map_lm(o.kinetic_eval(th2), start, np.zeros((1, 4, 4)), 0.0, 0.01, 60)[0]
    np.testing.assert_allclose(free[2], 0.05, rtol=1e-5)   # default box again: k3 is fitted
