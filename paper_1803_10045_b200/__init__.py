"""paper_1803_10045_b200 -- thin Python binding of libkcs.so (include/kcs.h).

Argument marshalling only: every step of the hot path (projection, Poisson ratio, back-projection, OSL update,
kinetic model, MAP-LM, the ICM sequencing) runs in the hand-written sm_100a kernels behind the C ABI.  PyTorch is
used for device memory and streams.  There is no CPU fallback: if libkcs.so is missing or no CUDA device is
present, the calls raise.

Names follow the C ABI: ``Context.forward_project`` <-> ``kcs_forward_project`` etc.; module-level aliases
``kcs_forward_project(ctx, ...)`` are provided too.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkcs.so")

KCS_OK = 0
ERRORS = {-1: "KCS_ERR_NULL", -2: "KCS_ERR_SHAPE", -3: "KCS_ERR_SUBSET", -4: "KCS_ERR_FRAMES", -5: "KCS_ERR_CUDA",
          -6: "KCS_ERR_ALLOC"}
PRIOR_POISSON_MATCHED = 0
PRIOR_ABSOLUTE = 1
R_PER_FRAME = 0
R_FULL = 1
MAX_FRAMES = 32
PEAK_PROBES = ("fp32_tflops", "fp64_tflops", "l2_gbs", "l1_gbs", "l2_gather_gbs")
PROFILE_CLASSES = ("pack", "unpack", "kinetic", "forward", "back", "lm", "other")

# every symbol include/kcs.h declares (tests/test_abi.py checks the library exports each of them)
EXPORTS = ["kcs_create", "kcs_destroy", "kcs_set_stream", "kcs_last_error", "kcs_workspace_bytes", "kcs_get_mask",
           "kcs_launch_count", "kcs_use_graphs", "kcs_graph_replays", "kcs_profile_enable", "kcs_profile_read", "kcs_forward_project", "kcs_back_project", "kcs_sensitivity", "kcs_osl_update",
           "kcs_kinetic_eval", "kcs_ki_map", "kcs_set_multiplicative", "kcs_set_fit_options", "kcs_map_lm", "kcs_icm_iteration", "kcs_icm_run", "kcs_icm_run_host",
           "kcs_forward_project_static", "kcs_static_last_error"]


class KcsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


class _Config(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("vx", C.c_float), ("vy", C.c_float), ("vz", C.c_float),
        ("n_angles", C.c_int), ("n_bins", C.c_int), ("bin_mm", C.c_float),
        ("n_steps", C.c_int), ("step_mm", C.c_float),
        ("n_subsets", C.c_int),
        ("n_frames", C.c_int),
        ("t_start_min", C.POINTER(C.c_double)), ("t_end_min", C.POINTER(C.c_double)),
        ("feng_A", C.c_float * 3), ("feng_lambda", C.c_float * 3),
        ("mask_host", C.POINTER(C.c_ubyte)),
        ("n_replicas", C.c_int),
    ]


class _FitOptions(C.Structure):
    _fields_ = [("frame_weights", C.POINTER(C.c_double)), ("neighbourhood", C.c_int), ("delta4", C.POINTER(C.c_double)),
                ("prior_curvature", C.c_int), ("box_lo", C.POINTER(C.c_double)), ("box_hi", C.POINTER(C.c_double))]


_lib = None


def load(build_if_missing: bool = True) -> C.CDLL:
    """dlopen libkcs.so (building it with nvcc first if it is missing or stale). Raises if that fails."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        from . import build as _b
        try:
            _b.build()
        except Exception as e:  # nvcc missing on the box: fall through to the existing .so, if any
            if not os.path.exists(LIB_PATH):
                raise RuntimeError(f"libkcs.so is missing and could not be built: {e}") from e
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found; run `python -m paper_1803_10045_b200.build` (no CPU fallback exists)")
    lib = C.CDLL(LIB_PATH)
    vp, fp, i, f = C.c_void_p, C.c_void_p, C.c_int, C.c_float
    lib.kcs_create.argtypes = [C.POINTER(vp), C.POINTER(_Config), vp]
    lib.kcs_destroy.argtypes = [vp]
    lib.kcs_set_stream.argtypes = [vp, vp]
    lib.kcs_last_error.argtypes = [vp]
    lib.kcs_last_error.restype = C.c_char_p
    lib.kcs_workspace_bytes.argtypes = [vp]
    lib.kcs_workspace_bytes.restype = C.c_longlong
    lib.kcs_launch_count.argtypes = [vp]
    lib.kcs_launch_count.restype = C.c_longlong
    lib.kcs_get_mask.argtypes = [vp, vp]
    lib.kcs_use_graphs.argtypes = [vp, i]
    lib.kcs_graph_replays.argtypes = [vp]
    lib.kcs_graph_replays.restype = C.c_longlong
    lib.kcs_profile_enable.argtypes = [vp, i]
    lib.kcs_profile_read.argtypes = [vp, vp, vp, i]
    lib.kcs_forward_project.argtypes = [vp, fp, fp, i, i, i]
    lib.kcs_back_project.argtypes = [vp, fp, fp, i, i, i]
    lib.kcs_sensitivity.argtypes = [vp, i, fp]
    lib.kcs_osl_update.argtypes = [vp, fp, fp, fp, fp, f, i, f]
    lib.kcs_kinetic_eval.argtypes = [vp, fp, fp, fp]
    lib.kcs_ki_map.argtypes = [vp, fp, fp]
    lib.kcs_set_multiplicative.argtypes = [vp, fp]
    lib.kcs_set_fit_options.argtypes = [vp, vp]
    lib.kcs_map_lm.argtypes = [vp, fp, fp, fp, f, f, i, fp]
    lib.kcs_icm_iteration.argtypes = [vp, fp, fp, i, f, fp, fp, fp, f, f, f, i]
    lib.kcs_icm_run.argtypes = [vp, fp, fp, i, f, fp, fp, fp, f, f, f, f, i, i]
    lib.kcs_icm_run_host.argtypes = [vp, fp, fp, i, f, fp, fp, fp, f, f, f, f, i, i]
    lib.kcs_forward_project_static.argtypes = [C.POINTER(_Config), fp, fp, i, i, vp]
    lib.kcs_static_last_error.argtypes = []
    lib.kcs_static_last_error.restype = C.c_char_p
    _lib = lib
    return lib


STATIC_SCRATCH_BYTES = 40 << 20  # KCS_STATIC_SCRATCH_BYTES of include/kcs.h


def forward_project_static(cfg: dict, x, y_s, subset: int = -1, stream=None):
    """kcs_forward_project_static: the forward projector without a Context and without any device allocation (its
    workspace is a static 40 MiB device array inside libkcs.so; larger geometries raise KCS_ERR_SHAPE).
    x [nf, nz, ny, nx] -> y_s [nf, nz, As, B] on `stream` (default: torch's current stream).  Calls share the array:
    calls that overlap on the GPU race."""
    lib = load()
    c = _Config()
    for k in ("nx", "ny", "nz", "n_angles", "n_bins", "n_steps", "n_subsets"):
        setattr(c, k, int(cfg[k]))
    for k in ("vx", "vy", "vz", "bin_mm", "step_mm"):
        setattr(c, k, float(cfg[k]))
    nf = int(x.shape[0])
    As = c.n_angles if subset < 0 else c.n_angles // max(c.n_subsets, 1)
    px, py = _dev(x, (nf, c.nz, c.ny, c.nx)), _dev(y_s, (nf, c.nz, As, c.n_bins))
    if stream is None:
        stream = _torch().cuda.current_stream().cuda_stream
    rc = lib.kcs_forward_project_static(C.byref(c), px, py, int(subset), nf, C.c_void_p(stream))
    if rc != KCS_OK:
        raise KcsError(rc, lib.kcs_static_last_error().decode())


def probe_peak(what: str, stream=None) -> float:
    """BENCH-ONLY (libkcs_probe.so, include/kcs_probe.h): measured machine peak 'fp32_tflops', 'fp64_tflops', 'l2_gbs',
    'l1_gbs' or 'l2_gather_gbs' on the current device."""
    from . import build as _b
    lib = C.CDLL(_b.build_probe())
    lib.kcs_probe_peak.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_void_p]
    lib.kcs_probe_last_error.restype = C.c_char_p
    out = C.c_double(0.0)
    if stream is None:
        stream = _torch().cuda.current_stream().cuda_stream
    if lib.kcs_probe_peak(PEAK_PROBES.index(what), C.byref(out), C.c_void_p(stream)) != 0:
        raise RuntimeError(lib.kcs_probe_last_error().decode())
    return float(out.value)


def _torch():
    import torch
    return torch


def _dev(t, shape=None):
    """Pointer of a contiguous fp32 CUDA tensor."""
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("expected a contiguous float32 CUDA tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return C.c_void_p(t.data_ptr())


class Context:
    """Owns one kcs_ctx.  cfg: dict with the keys of kcs_config (see kcs_inputs.config)."""

    def __init__(self, cfg: dict, mask: np.ndarray | None = None, stream=None):
        torch = _torch()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1803_10045_b200 needs a CUDA device (no CPU fallback exists)")
        self._lib = load()
        self.cfg = dict(cfg)
        ts = np.ascontiguousarray(cfg["t_start_min"], dtype=np.float64)
        te = np.ascontiguousarray(cfg["t_end_min"], dtype=np.float64)
        self._keep = (ts, te, None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8))
        c = _Config()
        for k in ("nx", "ny", "nz", "n_angles", "n_bins", "n_steps", "n_subsets"):
            setattr(c, k, int(cfg[k]))
        for k in ("vx", "vy", "vz", "bin_mm", "step_mm"):
            setattr(c, k, float(cfg[k]))
        c.n_frames = len(ts)
        c.t_start_min = ts.ctypes.data_as(C.POINTER(C.c_double))
        c.t_end_min = te.ctypes.data_as(C.POINTER(C.c_double))
        c.feng_A = (C.c_float * 3)(*cfg["feng_A"])
        c.feng_lambda = (C.c_float * 3)(*cfg["feng_lambda"])
        c.mask_host = None if mask is None else self._keep[2].ctypes.data_as(C.POINTER(C.c_ubyte))
        c.n_replicas = int(cfg.get("n_replicas", 1))
        self.n_replicas = max(1, c.n_replicas)
        self.nx, self.ny, self.nz = c.nx, c.ny, c.nz * self.n_replicas  # nz: all slices (replica-major)
        self.A, self.B, self.S, self.T = c.n_angles, c.n_bins, c.n_subsets, c.n_frames
        self.V = self.nx * self.ny * self.nz
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        self._h = C.c_void_p()
        rc = self._lib.kcs_create(C.byref(self._h), C.byref(c), C.c_void_p(stream))
        if rc != KCS_OK:
            raise KcsError(rc, self._lib.kcs_last_error(None).decode())

    # ---- plumbing -------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != KCS_OK:
            raise KcsError(rc, self._lib.kcs_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.kcs_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, stream):
        self._check(self._lib.kcs_set_stream(self._h, C.c_void_p(stream)))

    def workspace_bytes(self) -> int:
        return int(self._lib.kcs_workspace_bytes(self._h))

    def launch_count(self) -> int:
        return int(self._lib.kcs_launch_count(self._h))

    def use_graphs(self, on: bool = True):
        self._check(self._lib.kcs_use_graphs(self._h, int(bool(on))))

    def graph_replays(self) -> int:
        return int(self._lib.kcs_graph_replays(self._h))

    def profile_enable(self, on: bool = True):
        self._check(self._lib.kcs_profile_enable(self._h, int(bool(on))))

    def profile_read(self) -> dict:
        """{class name: (milliseconds, launches)} since the previous read (synchronises the stream)."""
        ms = np.zeros(len(PROFILE_CLASSES), dtype=np.float64)
        n = np.zeros(len(PROFILE_CLASSES), dtype=np.int64)
        self._check(self._lib.kcs_profile_read(self._h, ms.ctypes.data_as(C.c_void_p), n.ctypes.data_as(C.c_void_p),
                                               len(PROFILE_CLASSES)))
        return {k: (float(ms[q]), int(n[q])) for q, k in enumerate(PROFILE_CLASSES)}

    def mask(self) -> np.ndarray:
        m = np.zeros((self.ny, self.nx), dtype=np.uint8)
        self._check(self._lib.kcs_get_mask(self._h, m.ctypes.data_as(C.c_void_p)))
        return m

    def n_sub_angles(self, subset: int) -> int:
        return self.A if subset < 0 else self.A // self.S

    # ---- the six calls of BASELINE.json north_star (+ helpers) -----------------------------------
    def forward_project(self, x, y_s, subset: int = -1, f0: int = 0, nf: int | None = None):
        nf = self.T if nf is None else nf
        self._check(self._lib.kcs_forward_project(self._h, _dev(x, (self.T, self.nz, self.ny, self.nx)),
                                                  _dev(y_s, (self.T, self.nz, self.n_sub_angles(subset), self.B)),
                                                  subset, f0, nf))
        return y_s

    def back_project(self, q_s, b, subset: int = -1, f0: int = 0, nf: int | None = None):
        nf = self.T if nf is None else nf
        self._check(self._lib.kcs_back_project(self._h, _dev(q_s, (self.T, self.nz, self.n_sub_angles(subset), self.B)),
                                               _dev(b, (self.T, self.nz, self.ny, self.nx)), subset, f0, nf))
        return b

    def sensitivity(self, subset: int, sens):
        self._check(self._lib.kcs_sensitivity(self._h, subset, _dev(sens, (self.ny, self.nx))))
        return sens

    def osl_update(self, x, bp, sens, F, beta: float, prior_mode: int = PRIOR_POISSON_MATCHED, sigma2: float = 1.0):
        shp = (self.T, self.nz, self.ny, self.nx)
        self._check(self._lib.kcs_osl_update(self._h, _dev(x, shp), _dev(bp, shp), _dev(sens, (self.ny, self.nx)),
                                             _dev(F, shp), beta, prior_mode, sigma2))
        return x

    def kinetic_eval(self, theta, F, J=None):
        shp = (self.nz, self.ny, self.nx)
        self._check(self._lib.kcs_kinetic_eval(self._h, _dev(theta, (4,) + shp), _dev(F, (self.T,) + shp),
                                               None if J is None else _dev(J, (4, self.T) + shp)))
        return F

    def set_multiplicative(self, mult):
        """mult: float32 CUDA tensor [nz][A][B] (attenuation x normalisation factors) or None for unit factors."""
        self._check(self._lib.kcs_set_multiplicative(self._h, None if mult is None else _dev(mult, (self.nz, self.A, self.B))))

    def set_fit_options(self, frame_weights=None, neighbourhood: int = 6, delta4=None, prior_curvature: bool = False,
                        box_lo=None, box_hi=None):
        """kcs_fit_options: weighted least squares, the 3x3-clique neighbourhood (10), per-parameter Huber thresholds, Huber
        curvature in the LM matrix, another parameter box (lo == hi fixes a parameter); no arguments = defaults."""
        arr = lambda a, n: None if a is None else np.ascontiguousarray(a, dtype=np.float64)
        fw, d4, lo, hi = arr(frame_weights, self.T), arr(delta4, 4), arr(box_lo, 4), arr(box_hi, 4)
        assert fw is None or fw.size == self.T
        assert all(a is None or a.size == 4 for a in (d4, lo, hi))
        ptr = lambda a: None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))
        o = _FitOptions(ptr(fw), neighbourhood, ptr(d4), int(bool(prior_curvature)), ptr(lo), ptr(hi))
        self._check(self._lib.kcs_set_fit_options(self._h, C.byref(o)))

    def ki_map(self, theta, ki):
        shp = (self.nz, self.ny, self.nx)
        self._check(self._lib.kcs_ki_map(self._h, _dev(theta, (4,) + shp), _dev(ki, shp)))
        return ki

    def map_lm(self, x, theta, lam, gamma: float, delta: float, n_steps: int, cost=None):
        shp = (self.nz, self.ny, self.nx)
        self._check(self._lib.kcs_map_lm(self._h, _dev(x, (self.T,) + shp), _dev(theta, (4,) + shp), _dev(lam, shp),
                                         gamma, delta, n_steps, None if cost is None else _dev(cost, shp)))
        return theta

    def _r(self, r):
        if r.numel() == self.T:
            return R_PER_FRAME
        if r.numel() == self.T * self.nz * self.A * self.B:
            return R_FULL
        raise ValueError("r must have T or T*nz*A*B elements")

    def icm_iteration(self, y, r, scale: float, x, theta, lam, beta: float, gamma: float, delta: float, n_lm: int):
        shp = (self.nz, self.ny, self.nx)
        self._check(self._lib.kcs_icm_iteration(self._h, _dev(y, (self.T, self.nz, self.A, self.B)), _dev(r), self._r(r),
                                                scale, _dev(x, (self.T,) + shp), _dev(theta, (4,) + shp), _dev(lam, shp),
                                                beta, gamma, delta, n_lm))

    def icm_run(self, y, r, scale: float, x, theta, lam, beta_first: float, beta: float, gamma: float, delta: float,
                n_lm: int, n_iter: int):
        shp = (self.nz, self.ny, self.nx)
        self._check(self._lib.kcs_icm_run(self._h, _dev(y, (self.T, self.nz, self.A, self.B)), _dev(r), self._r(r),
                                          scale, _dev(x, (self.T,) + shp), _dev(theta, (4,) + shp), _dev(lam, shp),
                                          beta_first, beta, gamma, delta, n_lm, n_iter))

    def icm_run_host(self, y, r, scale: float, x, theta, lam, beta_first: float, beta: float, gamma: float, delta: float,
                     n_lm: int, n_iter: int):
        """HOST buffers: contiguous fp32 CPU tensors (pinned or not) or numpy arrays; x, theta, lam are updated in place."""
        def hp(a, n):
            if hasattr(a, "data_ptr"):
                assert not a.is_cuda and a.is_contiguous() and a.numel() == n and a.element_size() == 4
                return C.c_void_p(a.data_ptr())
            assert a.dtype == np.float32 and a.flags.c_contiguous and a.size == n
            return a.ctypes.data_as(C.c_void_p)
        nr = r.numel() if hasattr(r, "numel") else r.size
        r_mode = R_PER_FRAME if nr == self.T else R_FULL
        self._check(self._lib.kcs_icm_run_host(self._h, hp(y, self.T * self.nz * self.A * self.B), hp(r, nr), r_mode, scale,
                                               hp(x, self.T * self.V), hp(theta, 4 * self.V), hp(lam, self.V),
                                               beta_first, beta, gamma, delta, n_lm, n_iter))


def kcs_forward_project(ctx: Context, *a, **k):
    return ctx.forward_project(*a, **k)


def kcs_back_project(ctx: Context, *a, **k):
    return ctx.back_project(*a, **k)


def kcs_osl_update(ctx: Context, *a, **k):
    return ctx.osl_update(*a, **k)


def kcs_kinetic_eval(ctx: Context, *a, **k):
    return ctx.kinetic_eval(*a, **k)


def kcs_map_lm(ctx: Context, *a, **k):
    return ctx.map_lm(*a, **k)


def kcs_icm_iteration(ctx: Context, *a, **k):
    return ctx.icm_iteration(*a, **k)
