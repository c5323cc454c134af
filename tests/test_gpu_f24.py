"""SURVEY.md 8(f)2 / 8(f)4 on the GPU: kcs_set_fit_options (frame weights, 3x3-clique neighbourhood, per-parameter Huber
thresholds) against the oracle's kcso_set_lm_options."""
import numpy as np
import pytest

import kcs_inputs as ki
from oracle import Oracle

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
FLOORS = np.array([0.05, 0.05, 0.02, 0.02])


@pytest.fixture(autouse=True)
def _restore_oracle_defaults():
    yield
    Oracle.set_lm_options()


def _kcs():
    import paper_1803_10045_b200 as kcs
    return kcs


def dev(a):
    return torch.tensor(np.asarray(a), dtype=torch.float32, device="cuda").contiguous()


def host(t):
    return t.detach().cpu().numpy().astype(np.float64)


f32 = lambda a: np.float32(a).astype(np.float64)


def _lm_problem(cfg, o, seed, noise):
    mask = o.default_mask()
    _, th_true = ki.phantom(cfg)
    th_true = th_true * mask[None, None]
    x = o.kinetic_eval(th_true) * mask[None, None]
    rng = np.random.Generator(np.random.PCG64(seed))
    x = x * (1.0 + noise * rng.standard_normal(x.shape))
    return mask, f32(x), f32(ki.lm_start(th_true, seed + 1))


def _frac(thg, tho, mask):
    ok = np.abs(thg - tho) <= 1e-3 * np.maximum(np.abs(tho), FLOORS[:, None, None, None])
    return min(float(ok[p][:, mask > 0].mean()) for p in range(4))


@pytest.mark.parametrize("opts", [
    dict(frame_weights="durations"),                                             # weighted least squares alone
    dict(neighbourhood=10),                                                      # the 3x3 clique alone
    dict(delta4=[0.004, 0.02, 0.007, 0.011]),                                    # per-parameter thresholds alone
    dict(frame_weights="ramp", neighbourhood=10, delta4=[0.004, 0.02, 0.007, 0.011]),
    dict(prior_curvature=True),                                                  # Huber curvature in the LM matrix
    dict(box_lo=[0.0, 1e-4, 0.0, 0.0], box_hi=[2.0, 2.0, 0.0, 1.0]),             # k3 fixed at 0: the one-tissue model
    dict(neighbourhood=10, delta4=[0.004, 0.02, 0.007, 0.011], prior_curvature=True,
         box_lo=[0.01, 0.02, 0.0, 0.03], box_hi=[0.5, 1.0, 0.2, 0.03]),          # a tighter box, vB fixed at 0.03
])
def test_map_lm_with_fit_options(opts):
    cfg = ki.small_config(nx=45, ny=37, nz=3, n_angles=30, n_bins=51, n_subsets=5, n_steps=57, sched="C3")
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    T = cfg["n_frames"]
    opts = dict(opts)
    if opts.get("frame_weights") == "durations":     # weights proportional to the frame length (minutes)
        opts["frame_weights"] = np.asarray(cfg["t_end_min"]) - np.asarray(cfg["t_start_min"])
    elif opts.get("frame_weights") == "ramp":
        opts["frame_weights"] = np.concatenate([[0.0, 0.0], np.linspace(0.3, 2.0, T - 2)])   # two frames dropped
    mask, x, start = _lm_problem(cfg, o, 41, 0.1)
    lam0 = np.zeros(x.shape[1:])
    plain_th, plain_lam = dev(start), dev(lam0)
    ctx.map_lm(dev(x), plain_th, plain_lam, 3e5, 0.01, 3)
    Oracle.set_lm_options(frame_w=opts.get("frame_weights"), neighbourhood=opts.get("neighbourhood", 6), delta4=opts.get("delta4"),
                          prior_curvature=opts.get("prior_curvature", False), box_lo=opts.get("box_lo"), box_hi=opts.get("box_hi"))
    ctx.set_fit_options(**opts)
    for gamma in (0.0, 3e5):
        for n_steps in (1, 4):
            tho, lamo, costo = o.map_lm(x, start, lam0, gamma, 0.01, n_steps, want_cost=True)
            th, lam = dev(start), dev(lam0)
            cost = torch.zeros(x.shape[1:], dtype=torch.float32, device="cuda")
            ctx.map_lm(dev(x), th, lam, gamma, 0.01, n_steps, cost)
            assert _frac(host(th), tho, mask) >= 0.999, (gamma, n_steps)
            m = mask > 0
            assert np.mean(np.abs(host(cost)[:, m] - costo[:, m]) <= 1e-3 * np.abs(costo[:, m]) + 1e-6) >= 0.999
            assert np.mean(np.abs(host(lam)[:, m] - lamo[:, m]) <= 1e-3 * np.abs(lamo[:, m])) >= 0.999
    if "box_lo" in opts:                                     # fixed parameters sit exactly at their value
        for p in range(4):
            if opts["box_lo"][p] == opts["box_hi"][p]:
                assert np.all(host(th)[p][:, mask > 0] == np.float32(opts["box_lo"][p]))
    if "neighbourhood" in opts or "delta4" in opts or "prior_curvature" in opts:   # the options matter at gamma = 3e5
        assert not torch.equal(th, plain_th)
    ctx.set_fit_options()                                    # defaults: bit for bit the plain fit again
    th, lam = dev(start), dev(lam0)
    ctx.map_lm(dev(x), th, lam, 3e5, 0.01, 3)
    assert torch.equal(th, plain_th) and torch.equal(lam, plain_lam)
    ctx.close()


def test_icm_iteration_with_fit_options():
    cfg = ki.small_config(nx=32, ny=32, nz=2, n_angles=24, n_bins=32, n_subsets=4, counts=2e6)
    o = Oracle(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    x0, th0, r, scale = f32(x0), f32(th0), f32(prob["r"]), float(np.float32(prob["scale"]))
    w = np.asarray(cfg["t_end_min"]) - np.asarray(cfg["t_start_min"])
    d4 = [0.01, 0.02, 0.005, 0.005]
    Oracle.set_lm_options(frame_w=w, neighbourhood=10, delta4=d4)
    ctx = _kcs().Context(cfg)
    ctx.set_fit_options(frame_weights=w, neighbourhood=10, delta4=d4)
    xo, tho, lamo = x0, th0, lam0
    y, rd = dev(prob["y"]), dev(r)
    for beta in (0.0, 0.1):
        xs, ths, lams = dev(f32(xo)), dev(f32(tho)), dev(f32(lamo))
        xo, tho, lamo = o.icm_iteration(prob["y"], r, scale, f32(xo), f32(tho), f32(lamo), beta, 2e5, 0.01, 4)
        ctx.icm_iteration(y, rd, scale, xs, ths, lams, beta, 2e5, 0.01, 4)
        assert np.linalg.norm(host(xs) - xo) <= 1e-4 * np.linalg.norm(xo)
        assert _frac(host(ths), tho, mask) >= 0.999
    ctx.close()


def test_curvature_alone_is_one_newton_step_to_the_neighbour_mean():
    """The oracle's pin on the GPU: all frame weights 0, every difference inside delta, Huber curvature on -- one step puts
    every voxel on the mean of its (10) neighbours of the previous iterate, to fp32 rounding of the stored maps."""
    cfg = ki.small_config(nx=20, ny=18, nz=3, n_angles=8, n_bins=20, n_subsets=2)
    kcs = _kcs()
    ctx = kcs.Context(cfg, mask=np.ones((18, 20), dtype=np.uint8))
    T = cfg["n_frames"]
    rng = np.random.default_rng(5)
    prev = np.float32(np.array(ki.GREY)[:, None, None, None] * (1 + 0.01 * rng.uniform(-1, 1, size=(4, 3, 18, 20)))).astype(np.float64)
    ctx.set_fit_options(frame_weights=np.zeros(T), neighbourhood=10, delta4=[1.0] * 4, prior_curvature=True)
    th, lam = dev(prev), dev(np.zeros((3, 18, 20)))
    x = torch.ones((T, 3, 18, 20), dtype=torch.float32, device="cuda")
    ctx.map_lm(x, th, lam, 2.5, 0.0, 1)
    want = np.zeros_like(prev)
    cnt = np.zeros((3, 18, 20))
    for dz, dj, di in [(0, 0, -1), (0, 0, 1), (0, -1, 0), (0, 1, 0), (-1, 0, 0), (1, 0, 0), (0, -1, -1), (0, -1, 1), (0, 1, -1), (0, 1, 1)]:
        src = (slice(max(dz, 0), 3 + min(dz, 0)), slice(max(dj, 0), 18 + min(dj, 0)), slice(max(di, 0), 20 + min(di, 0)))
        dst = (slice(max(-dz, 0), 3 + min(-dz, 0)), slice(max(-dj, 0), 18 + min(-dj, 0)), slice(max(-di, 0), 20 + min(-di, 0)))
        want[(slice(None),) + dst] += prev[(slice(None),) + src]
        cnt[dst] += 1
    want /= cnt[None]
    np.testing.assert_allclose(host(th), want, rtol=2e-7)
    ctx.close()


def test_fit_option_errors():
    kcs = _kcs()
    cfg = ki.small_config()
    ctx = kcs.Context(cfg)
    with pytest.raises(kcs.KcsError) as e:
        ctx.set_fit_options(neighbourhood=8)
    assert e.value.code == -2
    with pytest.raises(kcs.KcsError) as e:
        ctx.set_fit_options(frame_weights=-np.ones(cfg["n_frames"]))
    assert e.value.code == -2
    with pytest.raises(kcs.KcsError) as e:
        ctx.set_fit_options(box_lo=[0.0, 0.5, 0.0, 0.0], box_hi=[1.0, 0.1, 1.0, 1.0])
    assert e.value.code == -2
    ctx.close()
