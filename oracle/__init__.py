"""ORACLE binding (test infrastructure, NOT the product).

ctypes wrapper around oracle/kcs_oracle.c -- the plain fp64 CPU statement of one ICM
iteration of Kinetic Compressive Sensing (arXiv 1803.10045).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It imports nothing from the CUDA package and vice versa.

All arrays are numpy float64, C order, layouts as in kcs_oracle.h.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kcs_oracle.c")
_HDR = os.path.join(_HERE, "kcs_oracle.h")
_LIB = os.path.join(_HERE, "libkcs_oracle.so")

PRIOR_POISSON_MATCHED = 0
PRIOR_ABSOLUTE = 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -fopenmp) if the .so is missing or stale."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(p) > os.path.getmtime(_LIB) for p in (_SRC, _HDR))
    if force or stale:
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=c11", "-shared", "-fPIC",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Cfg(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("vx", C.c_double), ("vy", C.c_double), ("vz", C.c_double),
        ("n_angles", C.c_int), ("n_bins", C.c_int), ("bin_mm", C.c_double),
        ("n_steps", C.c_int), ("step_mm", C.c_double),
        ("n_subsets", C.c_int),
        ("n_frames", C.c_int),
        ("t_start_min", C.POINTER(C.c_double)), ("t_end_min", C.POINTER(C.c_double)),
        ("feng_A", C.c_double * 3), ("feng_lambda", C.c_double * 3),
        ("mask", C.POINTER(C.c_ubyte)),
    ]


_lib = None


def _L():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        d, dp, vp = C.c_double, C.POINTER(C.c_double), C.c_void_p
        _lib.kcso_ICp.restype = d
        _lib.kcso_R.restype = d
        _lib.kcso_G.restype = d
        _lib.kcso_dGda.restype = d
        _lib.kcso_Ct.restype = d
        _lib.kcso_lm_objective.restype = d
        _lib.kcso_poisson_loglik.restype = d
        _lib.kcso_num_threads.restype = C.c_int
        _lib.kcso_get_lm_accept_slack.restype = d
        _lib.kcso_set_lm_accept_slack.argtypes = [d]
        _lib.kcso_ICp.argtypes = [vp, d]
        _lib.kcso_R.argtypes = [vp, d, d]
        _lib.kcso_G.argtypes = [vp, d, d]
        _lib.kcso_dGda.argtypes = [vp, d, d]
        _lib.kcso_Ct.argtypes = [vp, dp, d]
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def set_lm_accept_slack(s: float) -> float:
    """Q15a knob of the oracle (default 1e-6); returns the previous value."""
    old = float(_L().kcso_get_lm_accept_slack())
    _L().kcso_set_lm_accept_slack(float(s))
    return old


class Oracle:
    """One geometry + frame schedule + input function (kcso_config)."""

    def __init__(self, cfg: dict, mask: np.ndarray | None = None):
        """cfg keys: nx ny nz vx vy vz n_angles n_bins bin_mm n_steps step_mm n_subsets
        t_start_min t_end_min feng_A feng_lambda (see kcs_inputs.configs)."""
        self.cfg = dict(cfg)
        self._ts = _f64(cfg["t_start_min"]).copy()
        self._te = _f64(cfg["t_end_min"]).copy()
        self._mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
        c = _Cfg()
        for k in ("nx", "ny", "nz", "n_angles", "n_bins", "n_steps", "n_subsets"):
            setattr(c, k, int(cfg[k]))
        for k in ("vx", "vy", "vz", "bin_mm", "step_mm"):
            setattr(c, k, float(cfg[k]))
        c.n_frames = len(self._ts)
        c.t_start_min = _p(self._ts)
        c.t_end_min = _p(self._te)
        c.feng_A = (C.c_double * 3)(*cfg["feng_A"])
        c.feng_lambda = (C.c_double * 3)(*cfg["feng_lambda"])
        c.mask = None if self._mask is None else self._mask.ctypes.data_as(C.POINTER(C.c_ubyte))
        self._c = c
        self.nx, self.ny, self.nz = c.nx, c.ny, c.nz
        self.A, self.B, self.S, self.T = c.n_angles, c.n_bins, c.n_subsets, c.n_frames
        self.V = self.nx * self.ny * self.nz

    @property
    def ref(self):
        return C.byref(self._c)

    @staticmethod
    def num_threads() -> int:
        return int(_L().kcso_num_threads())

    def n_sub_angles(self, subset: int) -> int:
        return self.A if subset < 0 else self.A // self.S

    def default_mask(self) -> np.ndarray:
        m = np.zeros((self.ny, self.nx), dtype=np.uint8)
        _L().kcso_default_mask(self.ref, m.ctypes.data_as(C.POINTER(C.c_ubyte)))
        return m

    def mask(self) -> np.ndarray:
        return self.default_mask() if self._mask is None else self._mask.copy()

    # ---- projector -------------------------------------------------------------------------
    def forward_project(self, x: np.ndarray, subset: int = -1) -> np.ndarray:
        x = _f64(x).reshape(-1, self.nz, self.ny, self.nx)
        nf = x.shape[0]
        y = np.empty((nf, self.nz, self.n_sub_angles(subset), self.B))
        _L().kcso_forward_project(self.ref, _p(x), _p(y), C.c_int(subset), C.c_int(nf))
        return y

    def back_project(self, q: np.ndarray, subset: int = -1) -> np.ndarray:
        q = _f64(q).reshape(-1, self.nz, self.n_sub_angles(subset), self.B)
        nf = q.shape[0]
        b = np.empty((nf, self.nz, self.ny, self.nx))
        _L().kcso_back_project(self.ref, _p(q), _p(b), C.c_int(subset), C.c_int(nf))
        return b

    def sensitivity(self, subset: int = -1) -> np.ndarray:
        s = np.empty((self.ny, self.nx))
        _L().kcso_sensitivity(self.ref, C.c_int(subset), _p(s))
        return s

    def osl_update(self, x, bp, sens, F, beta, prior_mode=PRIOR_POISSON_MATCHED, sigma2=1.0):
        x = _f64(x).reshape(-1, self.nz, self.ny, self.nx).copy()
        nf = x.shape[0]
        bp, sens, F = _f64(bp), _f64(sens), _f64(F)
        assert bp.size == x.size and F.size == x.size and sens.size == self.nx * self.ny
        _L().kcso_osl_update(self.ref, _p(x), _p(bp), _p(sens), _p(F), C.c_double(beta),
                             C.c_int(prior_mode), C.c_double(sigma2), C.c_int(nf))
        return x

    # ---- kinetic model ---------------------------------------------------------------------
    def input_function(self, t) -> np.ndarray:
        t = _f64(np.atleast_1d(t))
        out = np.empty_like(t)
        _L().kcso_input_function(self.ref, _p(t), C.c_int(t.size), _p(out))
        return out

    def ICp(self, t: float) -> float:
        return float(_L().kcso_ICp(self.ref, float(t)))

    def R(self, a: float, t: float) -> float:
        return float(_L().kcso_R(self.ref, float(a), float(t)))

    def G(self, a: float, t: float) -> float:
        return float(_L().kcso_G(self.ref, float(a), float(t)))

    def dGda(self, a: float, t: float) -> float:
        return float(_L().kcso_dGda(self.ref, float(a), float(t)))

    def Ct(self, xi, t: float) -> float:
        xi = _f64(xi)
        return float(_L().kcso_Ct(self.ref, _p(xi), float(t)))

    def kinetic_eval(self, theta: np.ndarray, jac: bool = False):
        """theta[4, ...] -> F[T, ...] (and J[4, T, ...])."""
        theta = _f64(theta)
        shp = theta.shape[1:]
        V = int(np.prod(shp)) if shp else 1
        th = theta.reshape(4, V)
        F = np.empty((self.T, V))
        J = np.empty((4, self.T, V)) if jac else None
        _L().kcso_kinetic_eval(self.ref, _p(th), _p(F), _p(J), C.c_long(V))
        F = F.reshape((self.T,) + shp)
        if jac:
            return F, J.reshape((4, self.T) + shp)
        return F

    # ---- MAP-LM ----------------------------------------------------------------------------
    def lm_objective(self, xv, xi, nbr, gamma, delta) -> float:
        xv, xi = _f64(xv), _f64(xi)
        nbr = _f64(nbr).reshape(-1, 4)
        return float(_L().kcso_lm_objective(self.ref, _p(xv), _p(xi), _p(nbr), C.c_int(nbr.shape[0]),
                                            C.c_double(gamma), C.c_double(delta)))

    def map_lm(self, x, theta, lam, gamma, delta, n_steps, want_cost=False):
        x = _f64(x)
        theta = _f64(theta).reshape(4, self.nz, self.ny, self.nx).copy()
        lam = _f64(lam).reshape(self.nz, self.ny, self.nx).copy()
        assert x.size == self.T * self.V
        cost = np.zeros(self.V) if want_cost else None
        _L().kcso_map_lm(self.ref, _p(x), _p(theta), _p(lam), C.c_double(gamma), C.c_double(delta),
                         C.c_int(n_steps), _p(cost))
        if want_cost:
            return theta, lam, cost.reshape(self.nz, self.ny, self.nx)
        return theta, lam

    # ---- OS pass / ICM ---------------------------------------------------------------------
    def _r(self, r):
        r = _f64(r)
        if r.size == self.T:
            return r, 0
        assert r.size == self.T * self.nz * self.A * self.B
        return r, 1

    def os_pass(self, y, r, scale, x, F, beta, mult=None):
        """mult: multiplicative sinogram [nz][A][B] (attenuation x normalisation, S8(f)3), None = unity."""
        y, x, F = _f64(y), _f64(x).copy(), _f64(F)
        r, mode = self._r(r)
        if mult is None:
            _L().kcso_os_pass(self.ref, _p(y), _p(r), C.c_int(mode), C.c_double(scale), _p(x), _p(F), C.c_double(beta))
        else:
            mult = _f64(mult)
            assert mult.size == self.nz * self.A * self.B
            _L().kcso_os_pass_mult(self.ref, _p(y), _p(r), C.c_int(mode), C.c_double(scale), _p(mult), _p(x), _p(F),
                                   C.c_double(beta))
        return x.reshape(self.T, self.nz, self.ny, self.nx)

    def icm_iteration(self, y, r, scale, x, theta, lam, beta, gamma, delta, n_lm, mult=None):
        y, x = _f64(y), _f64(x).copy()
        theta, lam = _f64(theta).copy(), _f64(lam).copy()
        r, mode = self._r(r)
        if mult is None:
            _L().kcso_icm_iteration(self.ref, _p(y), _p(r), C.c_int(mode), C.c_double(scale), _p(x), _p(theta),
                                    _p(lam), C.c_double(beta), C.c_double(gamma), C.c_double(delta), C.c_int(n_lm))
        else:
            mult = _f64(mult)
            assert mult.size == self.nz * self.A * self.B
            _L().kcso_icm_iteration_mult(self.ref, _p(y), _p(r), C.c_int(mode), C.c_double(scale), _p(mult), _p(x), _p(theta),
                                         _p(lam), C.c_double(beta), C.c_double(gamma), C.c_double(delta), C.c_int(n_lm))
        return (x.reshape(self.T, self.nz, self.ny, self.nx),
                theta.reshape(4, self.nz, self.ny, self.nx), lam.reshape(self.nz, self.ny, self.nx))

    def icm_iteration_replicas(self, n_replicas, y, r, scale, x, theta, lam, beta, gamma, delta, n_lm):
        """N noise realisations of one object are N independent reconstructions.  Buffers are replica-major along z
        ([.., N*nz, ..]); this simply runs `icm_iteration` on each replica's slices in turn."""
        nz = self.nz
        y, x, theta, lam = _f64(y), _f64(x), _f64(theta), _f64(lam)
        y = y.reshape(self.T, n_replicas * nz, self.A, self.B)
        x = x.reshape(self.T, n_replicas * nz, self.ny, self.nx)
        theta = theta.reshape(4, n_replicas * nz, self.ny, self.nx)
        lam = lam.reshape(n_replicas * nz, self.ny, self.nx)
        xs, ths, lams = [], [], []
        for k in range(n_replicas):
            sl = slice(k * nz, (k + 1) * nz)
            a, b, c = self.icm_iteration(np.ascontiguousarray(y[:, sl]), r, scale, np.ascontiguousarray(x[:, sl]),
                                         np.ascontiguousarray(theta[:, sl]), np.ascontiguousarray(lam[sl]), beta, gamma, delta, n_lm)
            xs.append(a); ths.append(b); lams.append(c)
        return np.concatenate(xs, axis=1), np.concatenate(ths, axis=1), np.concatenate(lams, axis=0)

    @staticmethod
    def set_lm_options(frame_w=None, neighbourhood=6, delta4=None, prior_curvature=False, box_lo=None, box_hi=None):
        """S8(f)2 / S8(f)4: weighted least squares, the 3x3-clique neighbourhood (10), per-parameter Huber thresholds, Huber
        curvature in the LM matrix, another parameter box (lo == hi fixes a parameter).  Oracle-wide; call with no
        arguments to restore the defaults."""
        fw = None if frame_w is None else _f64(frame_w)
        d4 = None if delta4 is None else _f64(delta4)
        lo = None if box_lo is None else _f64(box_lo)
        hi = None if box_hi is None else _f64(box_hi)
        _L().kcso_set_lm_options(None if fw is None else _p(fw), C.c_int(0 if fw is None else fw.size), C.c_int(neighbourhood),
                                 None if d4 is None else _p(d4))
        _L().kcso_set_lm_options2(C.c_int(1 if prior_curvature else 0), None if lo is None else _p(lo), None if hi is None else _p(hi))

    @staticmethod
    def ki_map(theta):
        """K_i = K1 k3 / (k2 + k3)."""
        theta = _f64(theta)
        V = theta.size // 4
        ki = np.zeros(V)
        _L().kcso_ki_map(_p(theta), _p(ki), C.c_long(V))
        return ki.reshape(theta.shape[1:])

    def poisson_loglik(self, y, r, scale, x) -> float:
        y, x = _f64(y), _f64(x)
        r, mode = self._r(r)
        return float(_L().kcso_poisson_loglik(self.ref, _p(y), _p(r), C.c_int(mode), C.c_double(scale), _p(x)))
