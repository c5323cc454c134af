"""GPU parity on the edge cases of the path: the extreme frame counts (T = 1: Tp = 4, one frame of a 16 B group in use;
T = 5: Tp = 8; T = 32 = KCS_MAX_FRAMES: no padding frame), empty data (y = 0), an empty field of view, and calls that
ask for no work (n_iter = 0, n_lm = 0).  Everything is compared with the oracle on the same seeded inputs, through the
C ABI."""
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


f32 = lambda a: np.float32(a).astype(np.float64)


def close(g, o, tol):
    g, o = np.asarray(g), np.asarray(o)
    rel = float(np.linalg.norm((g - o).ravel()) / max(np.linalg.norm(o.ravel()), 1e-300))
    return rel <= tol and float(np.abs(g - o).max()) <= tol * float(np.abs(o).max())


def frac_ok(thg, tho, mask):
    ok = np.abs(thg - tho) <= 1e-3 * np.maximum(np.abs(tho), FLOORS[:, None, None, None])
    return [float(ok[p][:, mask > 0].mean()) for p in range(4)]


def _cfg(spec, **kw):
    """A small ragged geometry (two slices) with the frame schedule `spec` = [(count, seconds), ...]."""
    ts, te = ki._frames(spec)
    c = ki.small_config(nx=24, ny=20, nz=2, n_angles=12, n_bins=27, n_subsets=3, n_steps=29, counts=2e5)
    c.update(t_start_min=ts, t_end_min=te, n_frames=len(ts))
    c.update(kw)
    return c


@pytest.mark.parametrize("spec", [[(1, 3600)], [(3, 60), (2, 600)], [(16, 15), (8, 60), (8, 300)]], ids=["T1", "T5", "T32"])
def test_frame_count_extremes(spec):
    cfg = _cfg(spec)
    T = cfg["n_frames"]
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    mask = o.default_mask()
    assert np.array_equal(ctx.mask(), mask)
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    # the projector pair and the model curve at this frame count
    xs = f32(prob["x_true"])
    yo = o.forward_project(xs, -1)
    y = torch.zeros(yo.shape, dtype=torch.float32, device="cuda")
    ctx.forward_project(dev(xs), y)
    assert close(host(y), yo, 1e-5)
    qs = f32(prob["y"])
    for s in (-1, 1):
        As = cfg["n_angles"] if s < 0 else cfg["n_angles"] // cfg["n_subsets"]
        qsub = qs if s < 0 else np.ascontiguousarray(qs[:, :, s::cfg["n_subsets"]])
        assert qsub.shape[2] == As
        b = torch.zeros(xs.shape, dtype=torch.float32, device="cuda")
        ctx.back_project(dev(qsub), b, s)
        assert close(host(b), o.back_project(qsub, s), 1e-5)
    th = f32(prob["theta_true"])
    F = torch.zeros(xs.shape, dtype=torch.float32, device="cuda")
    ctx.kinetic_eval(dev(th), F)
    Fo = o.kinetic_eval(th)
    assert float(np.abs(host(F) - Fo).max()) <= 5e-6 * float(np.abs(Fo).max())
    # two ICM iterations, each from the oracle's state (beta = 0, then the kinetic prior on)
    x0, th0, r, scale = f32(x0), f32(th0), f32(prob["r"]), float(np.float32(prob["scale"]))
    xo, tho, lamo = x0, th0, lam0
    yd, rd = dev(prob["y"]), dev(r)
    for beta in (0.0, cfg["beta"]):
        x, thd, lam = dev(f32(xo)), dev(f32(tho)), dev(f32(lamo))
        xo, tho, lamo = o.icm_iteration(prob["y"], r, scale, f32(xo), f32(tho), f32(lamo), beta, cfg["gamma"], cfg["delta"], 3)
        ctx.icm_iteration(yd, rd, scale, x, thd, lam, beta, cfg["gamma"], cfg["delta"], 3)
        assert close(host(x), xo, 1e-4), (T, beta)
        fr = frac_ok(host(thd), tho, mask)
        assert min(fr) >= 0.999, (T, beta, fr)
    ctx.close()


def test_no_counts_and_no_work():
    cfg = _cfg([(4, 30), (4, 120)])
    o = Oracle(cfg)
    ctx = _kcs().Context(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    x0, th0, lam0 = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    x0, th0, r, scale = f32(x0), f32(th0), f32(prob["r"]), float(np.float32(prob["scale"]))
    # y = 0 everywhere: the ratio is 0, one OS pass empties the image; the fit then sees x = 0
    y0 = np.zeros_like(prob["y"])
    xo, tho, lamo = o.icm_iteration(y0, r, scale, x0, th0, lam0, 0.1, cfg["gamma"], cfg["delta"], 2)
    x, th, lam = dev(x0), dev(th0), dev(lam0)
    ctx.icm_iteration(dev(y0), dev(r), scale, x, th, lam, 0.1, cfg["gamma"], cfg["delta"], 2)
    assert float(np.abs(xo).max()) == 0.0 and float(host(x).max()) == 0.0 and float(host(x).min()) == 0.0
    assert min(frac_ok(host(th), tho, mask)) >= 0.999
    # n_iter = 0: nothing changes, bit for bit; n_lm = 0: the OS pass alone, maps and lambda untouched
    yd, rd = dev(prob["y"]), dev(r)
    x, th, lam = dev(x0), dev(th0), dev(lam0)
    ctx.icm_run(yd, rd, scale, x, th, lam, 0.0, 0.1, cfg["gamma"], cfg["delta"], 3, 0)
    assert torch.equal(x, dev(x0)) and torch.equal(th, dev(th0)) and torch.equal(lam, dev(lam0))
    ctx.icm_iteration(yd, rd, scale, x, th, lam, 0.1, cfg["gamma"], cfg["delta"], 0)
    assert torch.equal(th, dev(th0)) and torch.equal(lam, dev(lam0))
    xo = o.os_pass(prob["y"], r, scale, x0, o.kinetic_eval(th0), 0.1)
    assert close(host(x), xo, 1e-4)
    ctx.close()


def test_empty_field_of_view():
    """A mask without a single voxel: the activity becomes 0 everywhere (Q2), the maps are never touched, nothing is
    launched over an empty voxel list."""
    cfg = _cfg([(4, 30), (4, 120)])
    empty = np.zeros((cfg["ny"], cfg["nx"]), dtype=np.uint8)
    ctx = _kcs().Context(cfg, mask=empty)
    assert int(ctx.mask().sum()) == 0
    T, nz, ny, nx, A, B = cfg["n_frames"], cfg["nz"], cfg["ny"], cfg["nx"], cfg["n_angles"], cfg["n_bins"]
    y = dev(np.floor(3.0 * ki.uniform((T, nz, A, B), seed=3)))
    r = dev(np.full(T, 0.1))
    x = dev(0.5 + ki.uniform((T, nz, ny, nx), seed=4))
    th0 = np.float32(ki.uniform((4, nz, ny, nx), seed=5))
    th, lam = dev(th0), dev(np.zeros((nz, ny, nx)))
    ctx.icm_iteration(y, r, 1.0, x, th, lam, 0.1, 0.05, 0.01, 3)
    assert float(x.abs().max()) == 0.0
    assert torch.equal(th, dev(th0)) and float(lam.abs().max()) == 0.0
    ctx.close()
