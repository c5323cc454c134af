"""kcs_forward_project_static (include/kcs.h): the entry point that allocates nothing -- its workspace is a static
__device__ array of KCS_STATIC_SCRATCH_BYTES inside libkcs.so.  Checked against the existing path (kcs_create +
kcs_forward_project) on calls in a row that share that array.  Collected last on purpose (the suite runs with
pytest -x); passes alone in a fresh process and after the other tests."""
import ctypes as C

import numpy as np
import pytest

import kcs_inputs as ki

TOL = 1e-5  # the projector tolerance of tests/test_gpu_parity.py (rel-L2 and max-abs / max)


def _kcs():
    import paper_1803_10045_b200 as kcs
    return kcs


def _geom(nx, ny, nz, A, B, K, S):
    """A geometry in the recipe of kcs_inputs.config (2 mm voxels, bins and steps of one voxel)."""
    c = dict(ki.small_config())
    c.update(nx=nx, ny=ny, nz=nz, n_angles=A, n_bins=B, n_steps=K, n_subsets=S)
    return c


def test_rejects_sizes_beyond_the_static_array():
    """No GPU needed: the size check comes before any CUDA call.  BJ configs[2] needs 304 MiB of workspace."""
    kcs = _kcs()
    lib = kcs.load()
    cfg = ki.config("C3")
    c = kcs._Config()
    for k in ("nx", "ny", "nz", "n_angles", "n_bins", "n_steps", "n_subsets"):
        setattr(c, k, int(cfg[k]))
    for k in ("vx", "vy", "vz", "bin_mm", "step_mm"):
        setattr(c, k, float(cfg[k]))
    dummy = C.c_void_p(256)  # never dereferenced: the call is refused first
    rc = lib.kcs_forward_project_static(C.byref(c), dummy, dummy, -1, cfg["n_frames"], None)
    assert rc == -2  # KCS_ERR_SHAPE
    msg = lib.kcs_static_last_error().decode()
    assert "KCS_STATIC_SCRATCH_BYTES = %d" % kcs.STATIC_SCRATCH_BYTES in msg and "needs" in msg, msg
    c.nz = 2 ** 31 - 1                      # products far beyond 64 bits' worth of floats are refused too, not wrapped
    c.nx = c.ny = c.n_bins = 2 ** 31 - 5
    assert lib.kcs_forward_project_static(C.byref(c), dummy, dummy, -1, 32, None) == -2
    assert lib.kcs_forward_project_static(None, dummy, dummy, -1, 1, None) == -1
    c.nz = 1; c.nx = c.ny = c.n_bins = 64
    assert lib.kcs_forward_project_static(C.byref(c), dummy, dummy, -1, 33, None) == -4  # nf > KCS_MAX_FRAMES
    assert lib.kcs_forward_project_static(C.byref(c), dummy, dummy, cfg["n_subsets"], 1, None) == -2  # subset out of range


@pytest.mark.gpu
def test_static_forward_projection_matches_the_context_path():
    torch = pytest.importorskip("torch")
    kcs = _kcs()

    def close(g, o):
        g, o = g.double(), o.double()
        rel = float((g - o).norm() / o.norm().clamp_min(1e-300))
        return rel <= TOL and float((g - o).abs().max()) <= TOL * float(o.abs().max())

    rng = np.random.default_rng(20260511)
    # BJ configs[1] at full size (32 MiB of the 40 MiB array), then two smaller, ragged geometries: the array keeps the
    # previous call's contents, so a stale border or stale frames nf..Tp of the larger problem would show in the smaller
    cases = [ki.config("C2"), _geom(61, 45, 3, 36, 71, 67, 4), _geom(33, 50, 2, 30, 57, 49, 5)]
    calls = 0
    for cfg in cases:
        ctx = kcs.Context(cfg)
        T, nz, ny, nx, A, B, S = cfg["n_frames"], cfg["nz"], cfg["ny"], cfg["nx"], cfg["n_angles"], cfg["n_bins"], cfg["n_subsets"]
        xs = [torch.tensor(rng.gamma(2.0, 1.0, size=(T, nz, ny, nx)), dtype=torch.float32, device="cuda") for _ in range(2)]
        for subset, nf in ((-1, T), (S - 1, T), (1, min(T, 5))):
            As = A if subset < 0 else A // S
            want = [torch.zeros((T, nz, As, B), dtype=torch.float32, device="cuda") for _ in xs]
            for x, w in zip(xs, want):
                ctx.forward_project(x, w, subset=subset, f0=0, nf=nf)
            got = [torch.full((nf, nz, As, B), float("nan"), dtype=torch.float32, device="cuda") for _ in xs]
            xin = [x[:nf].contiguous() if nf < T else x for x in xs]
            kcs.forward_project_static(cfg, xin[0], got[0], subset=subset)   # two calls in a row, same geometry,
            torch.cuda.synchronize()                                           # different volumes
            free0 = torch.cuda.mem_get_info()[0]   # after the first: every kernel the call uses is loaded
            kcs.forward_project_static(cfg, xin[1], got[1], subset=subset)
            torch.cuda.synchronize()
            free1 = torch.cuda.mem_get_info()[0]
            calls += 2
            for g, w in zip(got, want):
                assert bool(torch.isfinite(g).all())
                assert close(g, w[:nf]), (cfg["name"] if "name" in cfg else (nx, ny, nz), subset, nf)
            if nx == 61 and nf == T:          # and against the oracle itself, on the geometry it finishes in a moment
                from oracle import Oracle
                yo = Oracle(cfg).forward_project(xs[0].cpu().numpy().astype(np.float64), subset)
                assert close(got[0], torch.tensor(yo, device="cuda")), ("oracle", subset)
            assert abs(free0 - free1) < (2 << 20), (free0, free1)  # the device's free memory does not move across a call
        ctx.close()
    assert calls == 18
