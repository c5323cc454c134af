"""Pins for the oracle's multiplicative sinogram ("all effects of attenuation, scatter and randoms"):
yhat = scale n (A x) + r, b = scale A^T (n q), S = scale A^T n, with n[nz][A][B] = attenuation x normalisation factors."""
import numpy as np

import kcs_inputs as ki
from oracle import Oracle
from test_oracle_projector import _dense_A


def _setup(nz=1, n_subsets=3, **kw):
    cfg = ki.small_config(nx=12, ny=10, nz=nz, n_angles=12, n_bins=14, n_subsets=n_subsets, n_steps=12, **kw)
    o = Oracle(cfg)
    rng = np.random.default_rng(3)
    T = cfg["n_frames"]
    mask = o.default_mask()
    x = rng.uniform(0.5, 2.0, (T, nz, 10, 12)) * mask[None, None]
    F = rng.uniform(0.5, 2.0, x.shape)
    y = rng.poisson(5.0, (T, nz, 12, 14)).astype(np.float64)
    r = rng.uniform(0.1, 0.5, T)
    n = rng.uniform(0.2, 1.0, (nz, 12, 14))            # attenuation factors e^{-mu l} in (0, 1]
    return cfg, o, mask, x, F, y, r, n


def test_unit_factors_are_the_plain_pass_and_uniform_factors_rescale():
    cfg, o, mask, x, F, y, r, n = _setup()
    plain = o.os_pass(y, r, 0.7, x, F, 0.1)
    assert np.array_equal(o.os_pass(y, r, 0.7, x, F, 0.1, mult=np.ones_like(n)), plain)
    # yhat = scale c (A x) + r, b / S = A^T(c q) / A^T c: a uniform factor c is the same as scale -> scale c
    np.testing.assert_allclose(o.os_pass(y, r, 0.7, x, F, 0.1, mult=np.full_like(n, 0.37)), o.os_pass(y, r, 0.7 * 0.37, x, F, 0.1),
                               rtol=1e-12, atol=1e-14)


def test_consistent_data_is_a_fixed_point_with_attenuation():
    cfg, o, mask, x, F, y, r, n = _setup()
    ybar = 0.7 * n[None] * o.forward_project(x) + r[:, None, None, None]
    out = o.os_pass(ybar, r, 0.7, x, F, 0.0, mult=n)
    np.testing.assert_allclose(out, x, rtol=1e-11, atol=1e-13)


def test_one_pass_against_the_dense_matrix():
    """S = 1: x <- x (M^T (n y / (s n M x + r))) / (M^T n) on the in-mask pixels, with M built entry by entry."""
    cfg, o, mask, x, F, y, r, n = _setup(n_subsets=1)
    M = _dense_A(cfg)
    s = 0.7
    got = o.os_pass(y, r, s, x, F, 0.0, mult=n)
    nv = n[0].ravel()
    S = s * (M.T @ nv)
    for t in range(cfg["n_frames"]):
        xt = x[t, 0].ravel()
        yh = s * nv * (M @ xt) + r[t]
        bp = s * (M.T @ (nv * y[t, 0].ravel() / yh))
        want = np.where(mask.ravel() > 0, xt * bp / S, 0.0)
        np.testing.assert_allclose(got[t, 0].ravel(), want, rtol=1e-11, atol=1e-13)


def test_sensitivity_is_per_slice():
    """Two slices with different factors: each equals the single-slice pass with its own n (prior included)."""
    cfg, o, mask, x, F, y, r, n = _setup(nz=2)
    both = o.os_pass(y, r, 0.7, x, F, 0.1, mult=n)
    o1 = Oracle(dict(cfg, nz=1))
    for z in range(2):
        one = o1.os_pass(y[:, z:z + 1], r, 0.7, x[:, z:z + 1], F[:, z:z + 1], 0.1, mult=n[z:z + 1])
        np.testing.assert_allclose(both[:, z:z + 1], one, rtol=1e-13, atol=1e-15)
    assert not np.allclose(both[:, 0], o1.os_pass(y[:, :1], r, 0.7, x[:, :1], F[:, :1], 0.1, mult=n[1:2]))
