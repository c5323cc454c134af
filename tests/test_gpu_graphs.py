"""launch-bound volumes replay their ICM iteration as a CUDA graph (kcs.h, kcs_use_graphs).  A replay must
give the bits of the direct launches, follow the buffers' current contents, and be dropped when an option changes."""
import numpy as np
import pytest

import kcs_inputs as ki
from oracle import Oracle

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _kcs():
    import paper_1803_10045_b200 as kcs
    return kcs


def dev(a):
    return torch.tensor(np.asarray(a), dtype=torch.float32, device="cuda").contiguous()


def _problem(**kw):
    cfg = ki.small_config(nx=45, ny=37, nz=3, n_angles=30, n_bins=51, n_subsets=5, n_steps=57, **kw)
    o = Oracle(cfg)
    mask = o.default_mask()
    prob = ki.make_problem(cfg, mask, o.kinetic_eval, o.forward_project, noisy=True)
    st = ki.initial_state(cfg, mask, prob["y"], prob["r"], prob["scale"], o.forward_project)
    return cfg, prob, st


def _run(ctx, cfg, prob, st, stream, n_calls, graphs, y2=None):
    """n_calls reconstructions of 2 iterations each into the SAME buffers (refilled between calls)."""
    outs = []
    with torch.cuda.stream(stream):
        ctx.use_graphs(graphs)
        y, r = dev(prob["y"]), dev(prob["r"])
        x, th, lam = dev(st[0]), dev(st[1]), dev(st[2])
        x0, th0, lam0 = x.clone(), th.clone(), lam.clone()
        for k in range(n_calls):
            x.copy_(x0); th.copy_(th0); lam.copy_(lam0)
            if y2 is not None and k == n_calls - 1:
                y.copy_(y2)                      # new DATA in the same buffer: a replay must read it
            ctx.icm_run(y, r, float(prob["scale"]), x, th, lam, 0.0, cfg["beta"], cfg["gamma"], cfg["delta"], 3, 2)
            outs.append((x.clone(), th.clone(), lam.clone()))
    stream.synchronize()
    return outs


def test_replay_equals_direct_launches_bit_for_bit():
    cfg, prob, st = _problem()
    side = torch.cuda.Stream()
    ctx = _kcs().Context(cfg, stream=side.cuda_stream)
    y2 = dev(ki.poisson(prob["ybar"], 77))
    n0 = ctx.launch_count()
    direct = _run(ctx, cfg, prob, st, side, 3, False, y2)
    n_direct = ctx.launch_count() - n0
    assert ctx.graph_replays() == 0
    n0 = ctx.launch_count()
    graph = _run(ctx, cfg, prob, st, side, 3, True, y2)
    assert ctx.graph_replays() == 2                              # call 1 captures, calls 2 and 3 replay
    assert ctx.launch_count() - n0 == n_direct                   # the launch count is what the graph holds
    for a, b in zip(direct, graph):
        assert all(torch.equal(p, q) for p, q in zip(a, b))
    assert not torch.equal(graph[0][0], graph[2][0])             # the third call saw the new data
    assert torch.equal(graph[0][0], graph[1][0])
    ctx.close()


def test_option_change_drops_the_graph_and_default_stream_falls_back():
    kcs = _kcs()
    cfg, prob, st = _problem()
    side = torch.cuda.Stream()
    ctx = kcs.Context(cfg, stream=side.cuda_stream)
    a = _run(ctx, cfg, prob, st, side, 2, True)
    assert ctx.graph_replays() == 1
    w = np.linspace(0.5, 1.5, cfg["n_frames"])
    ctx.set_fit_options(frame_weights=w)
    b = _run(ctx, cfg, prob, st, side, 2, True)                  # re-captured with the weighted fit
    assert ctx.graph_replays() == 2
    assert not torch.equal(a[0][1], b[0][1]) and torch.equal(b[0][1], b[1][1])
    ctx.use_graphs(False)
    with torch.cuda.stream(side):
        c = _run(ctx, cfg, prob, st, side, 1, False)
    assert torch.equal(c[0][1], b[0][1])
    ctx.close()
    # the legacy default stream cannot be captured: the call runs directly, same bits
    ctx0 = kcs.Context(cfg)
    d = _run(ctx0, cfg, prob, st, torch.cuda.default_stream(), 2, True)
    assert ctx0.graph_replays() == 0
    assert torch.equal(d[1][0], a[1][0]) and torch.equal(d[1][1], a[1][1])
    ctx0.close()


def test_large_volumes_are_not_captured():
    cfg = ki.small_config(nx=128, ny=128, nz=16, n_angles=24, n_bins=128, n_subsets=4, sched="C2", counts=1e7)
    assert cfg["nx"] * cfg["ny"] * cfg["nz"] * cfg["n_frames"] > 4e6
    kcs = _kcs()
    side = torch.cuda.Stream()
    ctx = kcs.Context(cfg, stream=side.cuda_stream)
    T = cfg["n_frames"]
    with torch.cuda.stream(side):
        y = torch.ones((T, 16, 24, 128), dtype=torch.float32, device="cuda")
        r = torch.full((T,), 0.1, dtype=torch.float32, device="cuda")
        m = dev(ctx.mask())
        x = (torch.ones((T, 16, 128, 128), dtype=torch.float32, device="cuda") * m).contiguous()
        th = (dev(np.array(ki.THETA0))[:, None, None, None] * m.expand(1, 16, 128, 128)).contiguous()
        lam = torch.zeros((16, 128, 128), dtype=torch.float32, device="cuda")
        for _ in range(2):
            ctx.icm_iteration(y, r, 1e-3, x, th, lam, 0.0, 0.05, 0.01, 1)
    side.synchronize()
    assert ctx.graph_replays() == 0 and bool(torch.isfinite(x).all())
    ctx.close()
