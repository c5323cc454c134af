"""Pins for the parts of the oracle that only show with nz > 1 (the z-direction of the 6-neighbourhood of L1/Q13, the
slice / frame offsets of the projector pair and of the OS pass) and the experiment behind reading Q15a.

None of these compares the oracle with itself through the same code path: the neighbour gathering is redone with numpy
indexing, the 3-D calls are compared with independent single-slice calls, and the symmetry test swaps two axes."""
import numpy as np
import pytest

import kcs_inputs as ki
import oracle as oracle_mod
from oracle import Oracle


def _vol_cfg(nx, ny, nz, **kw):
    return ki.small_config(nx=nx, ny=ny, nz=nz, n_angles=8, n_bins=max(nx, ny), n_subsets=2, **kw)


def _random_problem(cfg, seed):
    rng = np.random.default_rng(seed)
    shp = (cfg["nz"], cfg["ny"], cfg["nx"])
    base = np.array(ki.GREY)[:, None, None, None]
    th_true = base * (1 + 0.3 * rng.uniform(-1, 1, size=(4,) + shp))
    start = base * (1 + 0.3 * rng.uniform(-1, 1, size=(4,) + shp))
    o = Oracle(cfg, mask=np.ones((cfg["ny"], cfg["nx"]), dtype=np.uint8))
    x = o.kinetic_eval(th_true) * (1 + 0.05 * rng.standard_normal((cfg["n_frames"],) + shp))
    return o, x, start


def test_map_lm_cost_uses_the_six_neighbours_of_the_previous_iterate():
    """L1 / Q13: Phi_v after a step, as returned by kcso_map_lm, equals kcso_lm_objective evaluated with the
    neighbours gathered HERE by numpy indexing from the previous iterate (+-x, +-y, +-z, in-volume, in-mask).  gamma is
    large enough for the prior to dominate, so a wrong z stride, a swapped dz or a missed neighbour changes Phi by O(1)."""
    cfg = _vol_cfg(5, 6, 4)
    mask = np.ones((6, 5), dtype=np.uint8)
    mask[0, 0] = mask[5, 4] = mask[2, 3] = 0          # holes: out-of-mask neighbours must be skipped
    rng = np.random.default_rng(3)
    o_full, x, start = _random_problem(cfg, 3)
    o = Oracle(cfg, mask=mask)
    gamma, delta = 3e5, 0.01
    prev, lam = start * mask[None, None], np.zeros((4, 6, 5))
    for step in range(3):
        new, lam_new, cost = o.map_lm(x, prev, lam, gamma, delta, 1, want_cost=True)
        for z in range(4):
            for j in range(6):
                for i in range(5):
                    if not mask[j, i]:
                        assert cost[z, j, i] == 0.0
                        np.testing.assert_array_equal(new[:, z, j, i], prev[:, z, j, i])
                        continue
                    nb = []
                    for dz, dj, di in ((0, 0, -1), (0, 0, 1), (0, -1, 0), (0, 1, 0), (-1, 0, 0), (1, 0, 0)):
                        zz, jj, ii = z + dz, j + dj, i + di
                        if 0 <= zz < 4 and 0 <= jj < 6 and 0 <= ii < 5 and mask[jj, ii]:
                            nb.append(prev[:, zz, jj, ii])
                    ref = o.lm_objective(x[:, z, j, i], new[:, z, j, i], nb, gamma, delta)
                    assert abs(ref - cost[z, j, i]) <= 1e-11 * max(1.0, abs(ref)), (step, z, j, i)
        # the prior must matter in this test: dropping the z-neighbours changes the objective visibly
        z, j, i = 1, 3, 2
        nb4 = [prev[:, z, j + dj, i + di] for dj, di in ((0, -1), (0, 1), (-1, 0), (1, 0))]
        assert abs(o.lm_objective(x[:, z, j, i], new[:, z, j, i], nb4, gamma, delta) - cost[z, j, i]) > 1e-3 * cost[z, j, i]
        prev, lam = new, lam_new


def test_map_lm_is_symmetric_under_swapping_z_and_y():
    """With a full mask the fit only knows the lattice: swapping the z and y axes of every input must swap them in
    the output (the neighbour sum is re-ordered, so agreement is to rounding, not bitwise)."""
    cfg_a = _vol_cfg(4, 5, 3)
    cfg_b = _vol_cfg(4, 3, 5)
    o_a, x, start = _random_problem(cfg_a, 8)
    o_b = Oracle(cfg_b, mask=np.ones((3, 4), dtype=np.uint8))
    sw = lambda a: np.swapaxes(a, -3, -2).copy()
    for gamma in (0.0, 3e4):
        th_a, lam_a, cost_a = o_a.map_lm(x, start, np.zeros((3, 5, 4)), gamma, 0.01, 4, want_cost=True)
        th_b, lam_b, cost_b = o_b.map_lm(sw(x), sw(start), np.zeros((5, 3, 4)), gamma, 0.01, 4, want_cost=True)
        np.testing.assert_allclose(sw(th_b), th_a, rtol=1e-9, atol=1e-12)
        np.testing.assert_allclose(sw(cost_b), cost_a, rtol=1e-9)
        np.testing.assert_allclose(sw(lam_b), lam_a, rtol=1e-9)
    # and the symmetry is not vacuous: at gamma = 3e4 the z-neighbours change the result
    th_2d = np.stack([Oracle(_vol_cfg(4, 5, 1), mask=np.ones((5, 4), dtype=np.uint8)).map_lm(
        x[:, z:z + 1], start[:, z:z + 1], np.zeros((1, 5, 4)), 3e4, 0.01, 4)[0][:, 0] for z in range(3)], axis=1)
    assert np.abs(th_2d - th_a).max() > 1e-4


def test_large_gamma_pulls_to_the_mean_of_the_six_neighbours():
    """gamma huge, delta huge (quadratic prior), neighbours frozen: the minimiser of sum_k (xi - xi_k)^2 / 2 is the mean
    of the in-volume neighbours -- 6 of them for an interior voxel of a 3-D volume, z included."""
    cfg = _vol_cfg(5, 5, 3)
    o, x, frozen = _random_problem(cfg, 5)
    z, j, i = 1, 2, 2
    nbrs = [frozen[:, z, j, i - 1], frozen[:, z, j, i + 1], frozen[:, z, j - 1, i], frozen[:, z, j + 1, i],
            frozen[:, z - 1, j, i], frozen[:, z + 1, j, i]]
    cur, lam = frozen.copy(), np.zeros((3, 5, 5))
    for _ in range(80):
        new, lam = o.map_lm(x, cur, lam, 1e14, 10.0, 1)
        cur = frozen.copy()
        cur[:, z, j, i] = new[:, z, j, i]
    # the 1e-6 acceptance slack of Q15a lets the iterate stall within ~sqrt(1e-6) of the minimiser
    m6, m4 = np.mean(nbrs, axis=0), np.mean(nbrs[:4], axis=0)
    np.testing.assert_allclose(cur[:, z, j, i], m6, rtol=5e-4)
    assert (np.abs(m4 - m6) / m6).max() > 2e-2  # the z pair matters: the in-plane mean is 40x the tolerance away


@pytest.fixture(scope="module")
def stack3():
    cfg = ki.small_config(nx=12, ny=10, nz=3, n_angles=12, n_bins=14, n_subsets=3, n_steps=13)
    return cfg, Oracle(cfg), Oracle(dict(cfg, nz=1))


def test_projector_pair_3d_equals_stacked_slices(stack3):
    """P3: slices (and frames) are independent 2-D problems: the nz = 3, nf = 2 calls equal six single-slice calls."""
    cfg, o3, o1 = stack3
    rng = np.random.default_rng(0)
    x = rng.random((2, 3, 10, 12))
    for subset in (-1, 1):
        y3 = o3.forward_project(x, subset)
        As = o3.n_sub_angles(subset)
        q = rng.random((2, 3, As, 14))
        b3 = o3.back_project(q, subset)
        for f in range(2):
            for z in range(3):
                np.testing.assert_array_equal(y3[f, z], o1.forward_project(x[f, z][None, None], subset)[0, 0])
                np.testing.assert_array_equal(b3[f, z], o1.back_project(q[f, z][None, None], subset)[0, 0])
    # adjointness through the 3-D entry points too (a transposed z / frame offset on one side only would break it)
    y = o3.forward_project(x, -1)
    q = rng.random(y.shape)
    assert abs(np.vdot(y, q) - np.vdot(x, o3.back_project(q, -1))) <= 1e-12 * abs(np.vdot(y, q))


def test_os_pass_3d_equals_stacked_slices(stack3):
    """O1-O2 on a 3-slice volume with a full randoms sinogram equal three single-slice passes (frame / slice / angle
    offsets of y, r and F inside kcso_os_pass)."""
    cfg, o3, o1 = stack3
    rng = np.random.default_rng(1)
    T = cfg["n_frames"]
    x = rng.random((T, 3, 10, 12)) + 0.5
    F = rng.random((T, 3, 10, 12)) + 0.5
    y = rng.poisson(5.0, size=(T, 3, 12, 14)).astype(np.float64)
    r = rng.random((T, 3, 12, 14)) + 0.1
    out3 = o3.os_pass(y, r, 0.37, x, F, 0.1)
    for z in range(3):
        out1 = o1.os_pass(y[:, z:z + 1], r[:, z:z + 1], 0.37, x[:, z:z + 1], F[:, z:z + 1], 0.1)
        np.testing.assert_array_equal(out3[:, z], out1[:, 0])
    rt = rng.random(T) + 0.1                            # per-frame randoms: r[t] must go with frame t
    out3 = o3.os_pass(y, rt, 0.37, x, F, 0.1)
    full = np.broadcast_to(rt[:, None, None, None], y.shape).copy()
    np.testing.assert_array_equal(out3, o3.os_pass(y, full, 0.37, x, F, 0.1))


def _chain(o, cfg, prob, st, eps, seed):
    rng = np.random.default_rng(seed)
    x, th, lam = [a.copy() for a in st]
    for it in range(cfg["n_icm"]):
        x, th, lam = o.icm_iteration(prob["y"], prob["r"], prob["scale"], x, th, lam, 0.0 if it == 0 else cfg["beta"],
                                     cfg["gamma"], cfg["delta"], cfg["n_lm"])
        if eps > 0:
            x = x * (1 + eps * rng.standard_normal(x.shape))
    return x, th, lam


def test_Q15a_acceptance_slack_makes_the_icm_chain_well_posed():
    """The experiment behind reading Q15a, oracle against itself on C1, 10 ICM iterations: a 3e-8
    relative perturbation of x after every iteration (half an fp32 ulp) moves more than 1 % of the voxels by more than
    BASELINE's 1e-3 when the step is accepted on a bare `Phi_new <= Phi_old`, because converged voxels then accept or
    reject by coin flip and lambda follows; with the 1e-6 relative slack every voxel agrees."""
    cfg = ki.config("C1")
    o = Oracle(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    st = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    floors = np.array([0.05, 0.05, 0.02, 0.02])[:, None, None, None]
    m = mask > 0

    def lost(slack):
        old = oracle_mod.set_lm_accept_slack(slack)
        try:
            _, th_a, lam_a = _chain(o, cfg, prob, st, 0.0, 0)
            _, th_b, lam_b = _chain(o, cfg, prob, st, 3e-8, 1)
        finally:
            oracle_mod.set_lm_accept_slack(old)
        ok = np.abs(th_a - th_b) <= 1e-3 * np.maximum(np.abs(th_a), floors)
        lam_differs = np.abs(np.log10(np.maximum(lam_a, 1e-300) / np.maximum(lam_b, 1e-300)))[:, m] > 0.5
        return 1.0 - min(float(ok[p][:, m].mean()) for p in range(4)), float(lam_differs.mean())

    assert oracle_mod.set_lm_accept_slack(1e-6) == 1e-6   # the default the rest of the suite runs with
    lost_bare, lam_bare = lost(0.0)
    lost_slack, lam_slack = lost(1e-6)
    print("Q15a: voxels lost with a bare <=:", lost_bare, "(lambda differs in", lam_bare, "); with the slack:", lost_slack)
    assert lost_bare > 0.01 and lam_bare > 0.01
    assert lost_slack == 0.0 and lam_slack == 0.0
