"""SURVEY.md 8(f)1 on the GPU: N noise realisations batched through one context, the K_i epilogue, and
the three methods of P:156-160 as settings of the same ICM path -- against the oracle and against N single runs."""
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


def _batch_problem(n_rep, **kw):
    cfg = ki.small_config(nx=24, ny=20, nz=3, n_angles=12, n_bins=24, n_subsets=3, counts=6e5, **kw)
    o = Oracle(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=False)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["ybar"], prob["r"], prob["scale"], o.forward_project)
    y = ki.noise_realisations(prob["ybar"], cfg["seed"], n_rep)
    return cfg, o, mask, prob, y, f32(x0), f32(th0), lam0


def test_batched_replicas_equal_single_runs_bit_for_bit():
    """N realisations through one context with n_replicas = N give exactly what N separate contexts give: replicas share
    only geometry tables, and the Huber prior's z-neighbours stop at a replica's first and last slice (gamma is large here
    so that the prior decides the fit)."""
    n_rep = 3
    cfg, o, mask, prob, y, x0, th0, lam0 = _batch_problem(n_rep)
    nz, gamma = cfg["nz"], 2e5
    r, scale = dev(prob["r"]), float(prob["scale"])
    ctx = _kcs().Context(dict(cfg, n_replicas=n_rep))
    x, th, lam = (dev(ki.tile_replicas(x0, 1, n_rep)), dev(ki.tile_replicas(th0, 1, n_rep)), dev(ki.tile_replicas(lam0, 0, n_rep)))
    ctx.icm_run(dev(y), r, scale, x, th, lam, 0.0, cfg["beta"], gamma, cfg["delta"], 3, 3)
    one = _kcs().Context(cfg)
    for k in range(n_rep):
        sl = slice(k * nz, (k + 1) * nz)
        xs, ths, lams = dev(x0), dev(th0), dev(lam0)
        one.icm_run(dev(y[:, sl]), r, scale, xs, ths, lams, 0.0, cfg["beta"], gamma, cfg["delta"], 3, 3)
        assert torch.equal(xs, x[:, sl]) and torch.equal(ths, th[:, sl]) and torch.equal(lams, lam[sl]), k
    assert not torch.equal(x[:, :nz], x[:, nz:2 * nz])   # the realisations do differ
    ctx.close()
    one.close()


def test_batched_replicas_against_the_oracle():
    n_rep = 2
    cfg, o, mask, prob, y, x0, th0, lam0 = _batch_problem(n_rep)
    r, scale = f32(prob["r"]), float(np.float32(prob["scale"]))
    gamma = 3e5
    X0, TH0, L0 = ki.tile_replicas(x0, 1, n_rep), ki.tile_replicas(th0, 1, n_rep), ki.tile_replicas(lam0, 0, n_rep)
    xo, tho, lamo = o.icm_iteration_replicas(n_rep, y, r, scale, X0, TH0, L0, 0.0, gamma, cfg["delta"], 4)
    ctx = _kcs().Context(dict(cfg, n_replicas=n_rep))
    x, th, lam = dev(X0), dev(TH0), dev(L0)
    ctx.icm_iteration(dev(y), dev(r), scale, x, th, lam, 0.0, gamma, cfg["delta"], 4)
    assert np.linalg.norm(host(x) - xo) <= 1e-4 * np.linalg.norm(xo)
    assert np.abs(host(x) - xo).max() <= 1e-4 * np.abs(xo).max()
    ok = np.abs(host(th) - tho) <= 1e-3 * np.maximum(np.abs(tho), FLOORS[:, None, None, None])
    assert min(ok[p][:, mask > 0].mean() for p in range(4)) >= 0.999
    ctx.close()


def test_ki_map_against_the_oracle():
    cfg = ki.small_config(nx=64, ny=32, nz=2)
    ctx = _kcs().Context(cfg)
    rng = np.random.Generator(np.random.PCG64(5))
    th = np.stack([rng.uniform(0, 2, (2, 32, 64)), rng.uniform(1e-4, 2, (2, 32, 64)), rng.uniform(0, 1, (2, 32, 64)),
                   rng.uniform(0, 1, (2, 32, 64))])
    th[1:3, 0, 0, :8] = 0.0            # k2 + k3 = 0
    th[2, 1, 3, :] = 0.0               # k3 = 0: no trapping
    th = f32(th)
    kio = Oracle.ki_map(th)
    kig = torch.full((2, 32, 64), -1.0, dtype=torch.float32, device="cuda")
    ctx.ki_map(dev(th), kig)
    assert np.max(np.abs(host(kig) - kio) / np.maximum(np.abs(kio), 1e-6)) <= 1e-6
    assert np.all(host(kig)[0, 0, :8] == 0.0)
    ctx.close()


@pytest.mark.parametrize("method", ["INDIRECT", "DIRECT", "KCS"])
def test_three_methods_against_the_oracle(method):
    """P:156-160 as settings of one path (paper_1803_10045_b200/methods.py); the oracle runs the same sequence call by call.
    Two ICM iterations, three realisations, a Huber weight at which the prior matters."""
    from paper_1803_10045_b200 import methods
    n_rep = 2
    cfg, o, mask, prob, y, x0, th0, lam0 = _batch_problem(n_rep, n_icm=2, n_lm=3, gamma=2e5)
    r, scale = f32(prob["r"]), float(np.float32(prob["scale"]))
    X0, TH0, L0 = ki.tile_replicas(x0, 1, n_rep), ki.tile_replicas(th0, 1, n_rep), ki.tile_replicas(lam0, 0, n_rep)
    beta, gamma = {"INDIRECT": (0.0, 0.0), "DIRECT": (cfg["beta"], 0.0), "KCS": (cfg["beta"], cfg["gamma"])}[method]
    xo, tho, lamo = X0, TH0, L0
    for it in range(cfg["n_icm"]):
        n_lm = 0 if method == "INDIRECT" else cfg["n_lm"]
        xo, tho, lamo = o.icm_iteration_replicas(n_rep, y, r, scale, xo, tho, lamo, 0.0 if it == 0 else beta, gamma, cfg["delta"], n_lm)
    if method == "INDIRECT":
        nz = cfg["nz"]
        parts = [o.map_lm(xo[:, k * nz:(k + 1) * nz], tho[:, k * nz:(k + 1) * nz], lamo[k * nz:(k + 1) * nz], 0.0, cfg["delta"],
                          cfg["n_icm"] * cfg["n_lm"]) for k in range(n_rep)]
        tho = np.concatenate([p[0] for p in parts], axis=1)
    kio = Oracle.ki_map(tho)
    ctx = _kcs().Context(dict(cfg, n_replicas=n_rep))
    xg, thg, kig = methods.reconstruct(ctx, method, dev(y), dev(r), scale, dev(X0), dev(TH0), dev(L0), cfg)
    assert np.linalg.norm(host(xg) - xo) <= 2e-4 * np.linalg.norm(xo)      # two OS passes
    m = mask > 0
    ok = np.abs(host(kig) - kio) <= 1e-3 * np.maximum(np.abs(kio), 0.005)
    assert ok[:, m].mean() >= 0.999, ok[:, m].mean()
    ctx.close()


def test_methods_harness_runs_c1():
    from paper_1803_10045_b200 import methods
    out = methods.run("C1", n_replicas=4)
    assert set(out["methods"]) == {"INDIRECT", "DIRECT", "KCS"}
    for m, d in out["methods"].items():
        assert d["gpu_launches"] > 0
        for reg in ("white", "grey"):
            s = d["regions"][reg]
            assert np.isfinite(s["bias_pct"]) and np.isfinite(s["cov_pct"]) and s["cov_pct"] > 0.0
