"""Pins for the oracle's kinetic evaluator (pins table)."""
import os

import mpmath as mp
import numpy as np
import pytest

import kcs_inputs as ki
from oracle import Oracle

A1, A2, A3 = ki.FENG_A
L1, L2, L3 = ki.FENG_LAMBDA


@pytest.fixture(scope="module")
def o1():
    return Oracle(ki.config("C1"))


@pytest.fixture(scope="module")
def o3():
    return Oracle(ki.small_config(sched="C3"))


def test_input_function_golden(o1, golden_dir):
    for line in open(os.path.join(golden_dir, "feng_input_function.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kind, t, v = line.split()
        t, v = float(t), float(v)
        got = o1.input_function(t)[0] if kind == "cp" else o1.ICp(t)
        assert abs(got - v) <= 1e-11 * max(1.0, abs(v)), (kind, t)
    # the peak quoted in the golden file is a maximum
    tp = 0.289483644407
    assert o1.input_function(tp)[0] > o1.input_function(tp - 1e-3)[0]
    assert o1.input_function(tp)[0] > o1.input_function(tp + 1e-3)[0]


def test_tac_golden(o1, golden_dir):
    for line in open(os.path.join(golden_dir, "tac_c1_schedule.txt")):
        if line.startswith("#") or not line.strip():
            continue
        head, vals, ct40 = line.split("|")
        xi = np.array([float(v) for v in head.split()[1:]])
        ref = np.array([float(v) for v in vals.split()])
        F = o1.kinetic_eval(xi.reshape(4, 1))[:, 0]
        np.testing.assert_allclose(F, ref, rtol=2e-12)
        assert abs(o1.Ct(xi, 40.0) - float(ct40)) <= 1e-9


def _mp_Cp(t):
    return (A1 * t - A2 - A3) * mp.e ** (-L1 * t) + A2 * mp.e ** (-L2 * t) + A3 * mp.e ** (-L3 * t)


def _mp_Ct(xi, t):
    """The defining convolution K2 by adaptive quadrature (no closed form used)."""
    K1, k2, k3, vB = [mp.mpf(v) for v in xi]
    a = k2 + k3
    conv = mp.quad(lambda s: (K1 * k2 / a * mp.e ** (-a * (t - s)) + K1 * k3 / a) * _mp_Cp(s), [0, t])
    return vB * _mp_Cp(t) + (1 - vB) * conv


@pytest.mark.parametrize("xi", [ki.GREY, (0.07, 0.1091, 0.01, 0.1), (1.2, 1.5, 0.9, 0.4)])
def test_frame_integral_vs_nested_mpmath_quadrature(o1, xi):
    mp.mp.dps = 30
    F = o1.kinetic_eval(np.array(xi).reshape(4, 1))[:, 0]
    cfg = o1.cfg
    for m in (0, 3, 5, 11):
        ts, te = cfg["t_start_min"][m], cfg["t_end_min"][m]
        ref = mp.quad(lambda t: _mp_Ct(xi, t), [ts, te])
        assert abs(F[m] - float(ref)) <= 1e-9 * abs(float(ref)), m


def test_fine_grid_numerical_convolution(o3):
    """BASELINE north_star: closed-form TAC vs fine-grid (0.01 s) numerical convolution to 1e-8.
    Q22: 3-point Gauss-Legendre per 0.01 s cell; the exponential kernel makes the convolution an O(N) recursion."""
    h = 0.01 / 60.0
    t_end = float(o3.cfg["t_end_min"][-1])
    N = int(round(t_end / h))
    gl_x = np.array([-np.sqrt(0.6), 0.0, np.sqrt(0.6)]) * 0.5 + 0.5
    gl_w = np.array([5.0, 8.0, 5.0]) / 18.0
    edges = np.arange(N + 1) * h
    tq = edges[:-1, None] + gl_x[None, :] * h  # [N,3]
    Cp = o3.input_function(tq.ravel()).reshape(N, 3)
    for xi in (ki.GREY, ki.WHITE, ki.BACKGROUND, (0.5, 0.9, 0.3, 0.2)):
        K1, k2, k3, vB = xi
        a = k2 + k3
        # per cell: int_cell e^{-a(t1 - s)} Cp(s) ds and int_cell Cp
        cell_conv = h * (gl_w[None, :] * np.exp(-a * (edges[1:, None] - tq)) * Cp).sum(axis=1)
        cell_int = h * (gl_w[None, :] * Cp).sum(axis=1)
        R = np.zeros(N + 1)
        dec = np.exp(-a * h)
        for n in range(N):
            R[n + 1] = dec * R[n] + cell_conv[n]
        ICp = np.concatenate([[0.0], np.cumsum(cell_int)])
        tissue = K1 * k2 / a * R + K1 * k3 / a * ICp  # on cell edges
        Cp_e = o3.input_function(edges)
        Ct = vB * Cp_e + (1 - vB) * tissue
        # composite Simpson over edges (N even within every frame since frames are multiples of 0.02 s)
        F = o3.kinetic_eval(np.array(xi).reshape(4, 1))[:, 0]
        for m in range(o3.T):
            i0 = int(round(o3.cfg["t_start_min"][m] / h))
            i1 = int(round(o3.cfg["t_end_min"][m] / h))
            seg = Ct[i0:i1 + 1]
            simpson = h / 3.0 * (seg[0] + seg[-1] + 4 * seg[1:-1:2].sum() + 2 * seg[2:-1:2].sum())
            assert abs(simpson - F[m]) <= 1e-8 * abs(F[m]), (xi, m)


def test_ode_identity(o1):
    """R' = Cp - a R  =>  a G_a(t) = ICp(t) - R_a(t)."""
    for a in (1e-4, 0.0105, 0.1191, 0.15, 0.192, 1.0, 3.0):
        for t in (0.05, 0.5, 2.0, 10.0, 40.0):
            lhs = a * o1.G(a, t)
            rhs = o1.ICp(t) - o1.R(a, t)
            assert abs(lhs - rhs) <= 2e-10 * abs(o1.ICp(t)), (a, t)


def test_special_cases(o1):
    T = o1.T
    dICp = np.array([o1.ICp(te) - o1.ICp(ts) for ts, te in zip(o1.cfg["t_start_min"], o1.cfg["t_end_min"])])
    F = o1.kinetic_eval(np.array([0.1, 0.2, 0.05, 1.0]).reshape(4, 1))[:, 0]
    np.testing.assert_allclose(F, dICp, rtol=1e-13)  # vB = 1
    F = o1.kinetic_eval(np.array([0.0, 0.2, 0.05, 0.3]).reshape(4, 1))[:, 0]
    np.testing.assert_allclose(F, 0.3 * dICp, rtol=1e-13)  # K1 = 0
    # k3 = 0: one-tissue model, F = K1 * int_frame R_{k2}
    F = o1.kinetic_eval(np.array([0.1, 0.2, 0.0, 0.0]).reshape(4, 1))[:, 0]
    ref = [0.1 * (o1.G(0.2, te) - o1.G(0.2, ts)) for ts, te in zip(o1.cfg["t_start_min"], o1.cfg["t_end_min"])]
    np.testing.assert_allclose(F, ref, rtol=1e-13)
    mp.mp.dps = 30
    ts, te = o1.cfg["t_start_min"][5], o1.cfg["t_end_min"][5]
    one_tissue = mp.quad(lambda t: mp.quad(lambda s: 0.1 * mp.e ** (-0.2 * (t - s)) * _mp_Cp(s), [0, t]), [ts, te])
    assert abs(F[5] - float(one_tissue)) <= 1e-9 * F[5]
    # k2 -> small: pure trapping, tissue -> K1 * int Cp
    F = o1.kinetic_eval(np.array([0.1, 1e-12, 0.05, 0.0]).reshape(4, 1))[:, 0]
    ref = [0.1 * (o1.G(0.0, te) - o1.G(0.0, ts)) for ts, te in zip(o1.cfg["t_start_min"], o1.cfg["t_end_min"])]
    np.testing.assert_allclose(F, ref, rtol=1e-9)
    assert T == 12


def _mp_G(a, t):
    """K4 closed form in 40-digit arithmetic (valid away from a = lambda_i)."""
    a, t = mp.mpf(a), mp.mpf(t)
    s = 0
    for al, be, l in ((-A2 - A3, A1, L1), (A2, 0, L2), (A3, 0, L3)):
        l = mp.mpf(l)
        c = a - l
        P0 = lambda r: (1 - mp.e ** (-r * t)) / r if r != 0 else t
        P1 = (1 - mp.e ** (-l * t) * (1 + l * t)) / l ** 2
        d = P0(l) - P0(a)
        s += al * d / c + be * (P1 / c - d / c ** 2)
    return s


def test_continuity_across_lambda(o1):
    """Evaluate at lambda_i exactly and lambda_i +/- 1e-9 (removable singularity) against 40-digit values."""
    mp.mp.dps = 40
    for lam in (L2, L3, L1):
        for t in (0.5, 5.0, 30.0):
            ref_m = float(_mp_G(mp.mpf(lam) - mp.mpf("1e-9"), t))
            ref_p = float(_mp_G(mp.mpf(lam) + mp.mpf("1e-9"), t))
            for a, ref in ((lam - 1e-9, ref_m), (lam + 1e-9, ref_p), (lam, 0.5 * (ref_m + ref_p))):
                assert abs(o1.G(a, t) - ref) <= 1e-8 * abs(ref) + 1e-13, (lam, t, a)
            # switch-over points of the series/direct branches
            sw = 0.05
            for a in (lam + 0.995 * sw, lam + 1.005 * sw, lam - 0.995 * sw, lam - 1.005 * sw):
                if a <= 0:
                    continue
                ref = float(_mp_G(a, t))
                assert abs(o1.G(a, t) - ref) <= 1e-10 * abs(ref), (lam, t, a)


def test_dGda_vs_high_precision_difference(o1):
    mp.mp.dps = 40
    for a in (1e-3, 0.0105, 0.0603, 0.0692, 0.1191, 0.1192, 0.1690, 0.1692, 0.192, 0.5, 3.0, 4.13):
        for t in (0.1, 1.0, 10.0, 40.0):
            h = mp.mpf("1e-12")
            a_ = mp.mpf(a)
            if any(abs(a - l) < 1e-6 for l in (L1, L2, L3)):
                a_ = a_ + mp.mpf("1e-7")  # keep the closed form away from the pole
            ref = float((_mp_G(a_ + h, t) - _mp_G(a_ - h, t)) / (2 * h))
            assert abs(o1.dGda(float(a_), t) - ref) <= 1e-8 * abs(ref), (a, t)


@pytest.mark.parametrize("sched", ["C1", "C3"])
def test_jacobian_vs_central_differences(sched):
    o = Oracle(ki.small_config(sched=sched))
    rng = np.random.default_rng(3)
    pts = [ki.GREY, ki.WHITE, ki.BACKGROUND] + [tuple(rng.uniform([0.01, 0.02, 0.005, 0.0], [0.5, 0.6, 0.3, 0.3]))
                                                 for _ in range(5)]
    for xi in pts:
        xi = np.array(xi)
        F, J = o.kinetic_eval(xi.reshape(4, 1), jac=True)
        J = J[:, :, 0]
        for p in range(4):
            h = 1e-6
            xp, xm = xi.copy(), xi.copy()
            xp[p] += h
            xm[p] -= h
            num = (o.kinetic_eval(xp.reshape(4, 1))[:, 0] - o.kinetic_eval(xm.reshape(4, 1))[:, 0]) / (2 * h)
            scale = np.max(np.abs(num))
            assert np.max(np.abs(J[p] - num)) <= 1e-7 * scale + 1e-9, (xi, p)
