"""SURVEY.md 8(f)3 on the GPU: the multiplicative sinogram (attenuation x normalisation) through kcs_icm_*,
against the oracle's kcso_icm_iteration_mult."""
import numpy as np
import pytest

import kcs_inputs as ki
from oracle import Oracle

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
FLOORS = np.array([0.05, 0.05, 0.02, 0.02])


def _kcs():
    import paper_1803_10045_b200 as kcs
    return kcs


def dev(a):
    return torch.tensor(np.asarray(a), dtype=torch.float32, device="cuda").contiguous()


def host(t):
    return t.detach().cpu().numpy().astype(np.float64)


f32 = lambda a: np.float32(a).astype(np.float64)


def _problem(cfg, o, mult):
    """Data generated WITH the factors: y ~ Poisson(scale n A x_true + r)."""
    mask = o.default_mask()
    fwd_n = lambda x: mult[None] * o.forward_project(x)
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, fwd_n, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], fwd_n)
    return mask, prob, f32(x0), f32(th0), lam0


@pytest.mark.parametrize("name", ["ragged", "C2slab"])
def test_icm_iteration_with_attenuation(name):
    if name == "ragged":
        cfg = ki.small_config(nx=45, ny=37, nz=3, n_angles=30, n_bins=51, n_subsets=5, n_steps=57)
    else:  # C2's in-plane geometry and schedule (T = 24, 6 subsets), 2 slices
        cfg = dict(ki.config("C2"), nz=2, counts=8e6 * 2)
    o = Oracle(cfg)
    mult = f32(ki.attenuation_factors(cfg, o.forward_project))
    if name == "ragged":   # plus detector-efficiency (normalisation) factors that vary from bin to bin and slice to slice
        mult = f32(mult * ki.uniform(mult.shape, 91, 0.7, 1.0))
    assert 0.05 < mult.min() < 0.9 and mult.max() <= 1.0
    mask, prob, x0, th0, lam0 = _problem(cfg, o, mult)
    r, scale = f32(prob["r"]), float(np.float32(prob["scale"]))
    ctx = _kcs().Context(cfg)
    y, rd = dev(prob["y"]), dev(r)
    plain = [dev(x0), dev(th0), dev(lam0)]
    ctx.icm_iteration(y, rd, scale, *plain, 0.0, cfg["gamma"], cfg["delta"], 3)
    ctx.set_multiplicative(dev(mult))
    xo, tho, lamo = x0, th0, lam0
    x, th, lam = dev(x0), dev(th0), dev(lam0)
    for beta in (0.0, cfg["beta"]):
        xs, ths, lams = dev(f32(xo)), dev(f32(tho)), dev(f32(lamo))      # each iteration from the oracle's state
        xo, tho, lamo = o.icm_iteration(prob["y"], r, scale, f32(xo), f32(tho), f32(lamo), beta, cfg["gamma"], cfg["delta"], 3, mult=mult)
        ctx.icm_iteration(y, rd, scale, xs, ths, lams, beta, cfg["gamma"], cfg["delta"], 3)
        xg = host(xs)
        assert np.linalg.norm(xg - xo) <= 1e-4 * np.linalg.norm(xo), beta
        assert np.abs(xg - xo).max() <= 1e-4 * np.abs(xo).max(), beta
        ok = np.abs(host(ths) - tho) <= 1e-3 * np.maximum(np.abs(tho), FLOORS[:, None, None, None])
        assert min(ok[p][:, mask > 0].mean() for p in range(4)) >= 0.999, beta
    # the host-buffer entry (z chunks) takes the same factors
    hx, hth, hlam = np.float32(x0), np.float32(th0), np.float32(lam0)
    ctx.icm_iteration(y, rd, scale, x, th, lam, 0.0, cfg["gamma"], cfg["delta"], 3)
    ctx.icm_run_host(np.float32(prob["y"]), np.float32(r), scale, hx, hth, hlam, 0.0, 0.0, cfg["gamma"], cfg["delta"], 3, 1)
    assert np.array_equal(hx, x.cpu().numpy()) and np.array_equal(hth, th.cpu().numpy())
    # attenuation changes the result, and NULL restores the plain operator bit for bit
    assert not torch.equal(x, plain[0])
    ctx.set_multiplicative(None)
    again = [dev(x0), dev(th0), dev(lam0)]
    ctx.icm_iteration(y, rd, scale, *again, 0.0, cfg["gamma"], cfg["delta"], 3)
    assert all(torch.equal(a, b) for a, b in zip(again, plain))
    ctx.close()


def test_unit_factors_match_the_plain_path():
    cfg = ki.small_config(nx=24, ny=20, nz=2, n_angles=12, n_bins=24, n_subsets=3)
    o = Oracle(cfg)
    mask, prob, x0, th0, lam0 = _problem(cfg, o, np.ones((2, 12, 24)))
    ctx = _kcs().Context(cfg)
    y, rd, scale = dev(prob["y"]), dev(prob["r"]), float(prob["scale"])
    a = [dev(x0), dev(th0), dev(lam0)]
    ctx.icm_iteration(y, rd, scale, *a, 0.1, cfg["gamma"], cfg["delta"], 2)
    ctx.set_multiplicative(torch.ones((2, 12, 24), dtype=torch.float32, device="cuda"))
    b = [dev(x0), dev(th0), dev(lam0)]
    ctx.icm_iteration(y, rd, scale, *b, 0.1, cfg["gamma"], cfg["delta"], 2)
    # the sensitivity comes from a back-projection of ones instead of the fp64 table sum: equal to fp32 rounding
    assert np.linalg.norm(host(a[0]) - host(b[0])) <= 2e-6 * np.linalg.norm(host(a[0]))
    ctx.close()
