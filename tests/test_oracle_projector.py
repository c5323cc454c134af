"""Pins for the oracle's projector pair (pins table row "Projector pair")."""
import math

import numpy as np
import pytest

import kcs_inputs as ki
from oracle import Oracle


def _dense_A(cfg):
    """Brute force: the system matrix of P1-P3 built entry by entry with pure-Python loops (tiny sizes)."""
    nx, ny, A, B, K = cfg["nx"], cfg["ny"], cfg["n_angles"], cfg["n_bins"], cfg["n_steps"]
    M = np.zeros((A * B, ny * nx))
    for a in range(A):
        th = math.pi * a / A
        for b in range(B):
            s = (b - (B - 1) / 2) * cfg["bin_mm"]
            for k in range(K):
                u = (k - (K - 1) / 2) * cfg["step_mm"]
                fx = (s * math.cos(th) - u * math.sin(th)) / cfg["vx"] + (nx - 1) / 2
                fy = (s * math.sin(th) + u * math.cos(th)) / cfg["vy"] + (ny - 1) / 2
                for j in range(ny):
                    for i in range(nx):
                        w = max(0.0, 1 - abs(fx - i)) * max(0.0, 1 - abs(fy - j))  # tent x tent (P4)
                        if w:
                            M[a * B + b, j * nx + i] += cfg["step_mm"] * w
    return M


def test_brute_force_matrix_tiny():
    cfg = ki.small_config(nx=7, ny=6, n_angles=8, n_bins=9, n_subsets=2, n_steps=8)
    o = Oracle(cfg)
    M = _dense_A(cfg)
    rng = np.random.default_rng(1)
    x = rng.random((1, 1, 6, 7))
    q = rng.random((1, 1, 8, 9))
    np.testing.assert_allclose(o.forward_project(x).ravel(), M @ x.ravel(), rtol=0, atol=1e-12)
    np.testing.assert_allclose(o.back_project(q).ravel(), M.T @ q.ravel(), rtol=0, atol=1e-12)
    # subsets: a mod S == s (P5)
    for s in range(2):
        rows = np.concatenate([np.arange(a * 9, (a + 1) * 9) for a in range(s, 8, 2)])
        np.testing.assert_allclose(o.forward_project(x, s).ravel(), M[rows] @ x.ravel(), atol=1e-12)
        qs = rng.random((1, 1, 4, 9))
        np.testing.assert_allclose(o.back_project(qs, s).ravel(), M[rows].T @ qs.ravel(), atol=1e-12)
        np.testing.assert_allclose(o.sensitivity(s).ravel(), M[rows].sum(axis=0), atol=1e-12)


@pytest.mark.parametrize("name", ["C1"])
def test_adjointness(name):
    """<A x, y> = <x, A^T y> to 1e-10 relative (BASELINE.json north_star)."""
    cfg = ki.config(name)
    o = Oracle(cfg)
    rng = np.random.default_rng(0)
    x = rng.random((3, cfg["nz"], cfg["ny"], cfg["nx"]))
    y = rng.random((3, cfg["nz"], cfg["n_angles"], cfg["n_bins"]))
    lhs = float((o.forward_project(x) * y).sum())
    rhs = float((x * o.back_project(y)).sum())
    assert abs(lhs - rhs) <= 1e-10 * abs(lhs)
    for s in (0, cfg["n_subsets"] - 1):
        ys = rng.random((3, cfg["nz"], cfg["n_angles"] // cfg["n_subsets"], cfg["n_bins"]))
        lhs = float((o.forward_project(x, s) * ys).sum())
        rhs = float((x * o.back_project(ys, s)).sum())
        assert abs(lhs - rhs) <= 1e-10 * abs(lhs)


def test_axis_aligned_closed_form():
    """theta = 0 and 90 deg with B = nx, bin = step = voxel: samples fall on pixel centres, so
    (A f)[0][b] = step * column sums and (A f)[A/2][b] = step * row sums, exactly."""
    cfg = ki.small_config(nx=16, ny=16, n_angles=12, n_bins=16, n_subsets=3)
    o = Oracle(cfg)
    f = np.random.default_rng(2).random((1, 1, 16, 16))
    y = o.forward_project(f)[0, 0]
    np.testing.assert_allclose(y[0], cfg["step_mm"] * f[0, 0].sum(axis=0), rtol=0, atol=1e-12)
    # theta = 90 deg: X = -u, Y = s  -> bin b reads row b; (cos(pi/2) is 6e-17, not 0: tolerance covers it)
    np.testing.assert_allclose(y[6], cfg["step_mm"] * f[0, 0].sum(axis=1), rtol=0, atol=1e-10)


def test_impulse_row_equals_column():
    cfg = ki.small_config(nx=12, ny=12, n_angles=8, n_bins=12, n_subsets=2)
    o = Oracle(cfg)
    e = np.zeros((1, 1, 12, 12))
    e[0, 0, 7, 4] = 1.0
    col = o.forward_project(e)[0, 0]  # column of A
    for (a, b) in [(0, 4), (3, 6), (5, 5)]:
        g = np.zeros((1, 1, 8, 12))
        g[0, 0, a, b] = 1.0
        assert abs(o.back_project(g)[0, 0, 7, 4] - col[a, b]) < 1e-14


def test_disc_chord_length():
    """Centred disc of radius rho: (A f)(s) -> 2 sqrt(rho^2 - s^2) within O(voxel) (sanity)."""
    cfg = ki.small_config(nx=64, ny=64, n_angles=6, n_bins=64, n_subsets=1)
    o = Oracle(cfg)
    X = (np.arange(64) - 31.5) * 2.0
    rho = 40.0
    f = ((X[None, :] ** 2 + X[:, None] ** 2) <= rho * rho).astype(float)[None, None]
    y = o.forward_project(f)[0, 0]
    chord = 2 * np.sqrt(np.maximum(rho * rho - X * X, 0.0))
    inner = np.abs(X) < rho - 6
    assert np.max(np.abs(y[:, inner] - chord[None, inner])) < 2.5 * cfg["vx"]


def test_default_mask_counts():
    """Q2 mask; in-FOV voxel counts quoted in SURVEY.md 8 table (3 024 for C1, 99 936 for C2)."""
    assert int(Oracle(ki.config("C1")).default_mask().sum()) == 3024
    assert int(Oracle(ki.config("C2")).default_mask().sum()) * 8 == 99936


def test_q23_samples_on_pixel_centres_leave_no_residue_on_the_neighbours():
    """Reading Q23.  At 0 and 90 degrees with bin = step = voxel every sample of P2 lies exactly on a pixel centre, so in
    exact arithmetic one sinogram bin back-projects onto ONE image column (row) and nothing else.  With the mMR voxel size
    2.09 mm the index fx = X / vx + (nx - 1)/2 carries ~1e-14 of rounding for some bins (b = 48 of 344 is one); without the
    snap that leaves a weight of 1.4e-14 on the neighbouring column, which a noise-dominated OSL update amplifies by 20
    orders of magnitude within one pass (Q23).  Pin (C4's in-plane geometry): the back-projection of
    ANY single bin at those two angles is exactly step_mm on its column / row and EXACTLY zero everywhere else; the
    brute-force tent matrix (test_brute_force_matrix_tiny) still matches to 1e-12, i.e. the snap moves no weight by more
    than 1e-9."""
    n, A = 344, 252
    cfg = ki.small_config(nx=n, ny=n, n_angles=A, n_bins=n, n_subsets=21, n_steps=n, vx=2.09, vy=2.09, bin_mm=2.09, step_mm=2.09)
    o = Oracle(cfg)
    bins = [3, 46, 47, 48, 171, 172, 300, 343]
    for a, axis in ((0, "column"), (A // 2, "row")):
        q = np.zeros((len(bins), 1, A, n))           # "frame" f holds the unit sinogram of bin bins[f]
        q[np.arange(len(bins)), 0, a, bins] = 1.0
        img = o.back_project(q)[:, 0]                # [f][ny][nx]
        for f, b in enumerate(bins):
            want = np.zeros((n, n))
            if axis == "column":
                want[:, b] = cfg["step_mm"]          # theta = 0: X = s_b, the ray runs along y through column b
            else:
                want[b, :] = cfg["step_mm"]          # theta = 90 degrees: Y = s_b, the ray runs along x through row b
            assert np.count_nonzero(img[f]) == n, (a, b, np.count_nonzero(img[f]))
            assert np.array_equal(img[f], want), (a, b)
    # forward: the same columns / rows (sums of n pixels times step)
    x = np.random.default_rng(5).random((1, 1, n, n))
    y = o.forward_project(x)[0, 0]
    np.testing.assert_allclose(y[0], cfg["step_mm"] * x[0, 0].sum(axis=0), rtol=1e-13)
    np.testing.assert_allclose(y[A // 2], cfg["step_mm"] * x[0, 0].sum(axis=1), rtol=1e-13)
