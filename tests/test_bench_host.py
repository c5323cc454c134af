"""Host logic of bench.py that needs no GPU: the algorithmic work model and the max-rule
roofline (T_lb = max(HBM, L2, FMA), frac = T_lb / measured)."""
import numpy as np
import pytest

import bench
import kcs_inputs as ki


def _disc_mask(cfg):
    n = min(cfg["nx"], cfg["ny"], cfg["n_bins"], cfg["n_steps"])
    rad = (0.5 * n - 1.0) * cfg["vx"]
    X = (np.arange(cfg["nx"]) - 0.5 * (cfg["nx"] - 1)) * cfg["vx"]
    Y = (np.arange(cfg["ny"]) - 0.5 * (cfg["ny"] - 1)) * cfg["vy"]
    return (X[None, :] ** 2 + Y[:, None] ** 2 <= rad * rad).astype(np.uint8)


def test_work_model_matches_survey_table():
    """sample-frames per full forward 2.95e6 / 3.77e8 / 5.11e9 / 1.098e11; in-FOV voxels (Q2)."""
    want = {"C1": (2.95e6, 3024), "C2": (3.77e8, 99936), "C3": (5.11e9, 799488), "C4": (1.098e11, 11666220)}
    for name, (sf, vin) in want.items():
        cfg = ki.config(name)
        m = _disc_mask(cfg)
        assert int(m.sum()) * cfg["nz"] == vin
        wm = bench.work_model(cfg, m)
        assert wm["forward"]["units_defined"] * cfg["n_subsets"] == pytest.approx(sf, rel=5e-3)
        assert wm["back"]["units_defined"] * cfg["n_subsets"] == pytest.approx(sf, rel=5e-3)  # B K = nx ny
        # clipping to the field of view can only remove work, and not more than the corners of the square
        assert 0.75 * wm["forward"]["units_defined"] < wm["forward"]["units"] <= wm["forward"]["units_defined"]
        assert wm["forward"]["flops"] == 8.0 * wm["forward"]["units"] and wm["forward"]["l2_bytes"] == 4.0 * wm["forward"]["units"]
        assert wm["back"]["flops"] == 6.0 * wm["back"]["units"]
        full = bench.work_model(cfg, m, subset=False, clipped=False)
        assert full["forward"]["units"] == full["forward"]["units_defined"] == pytest.approx(sf, rel=5e-3)


def test_roofline_takes_the_binding_term():
    peaks = {"hbm_gbs": 6500.0, "l2_gbs": 17000.0, "fp32_tflops": 64.0}
    w = {"units": 1e9, "units_defined": 1e9, "unit": "u", "flops": 8e9, "l2_bytes": 4e9, "hbm_bytes": 3e7}
    r = bench.bounds(w, 1.0, peaks)
    t = r["t_bound_ms"]
    assert t["l2"] == pytest.approx(4e9 / 17e12 * 1e3) and t["alu"] == pytest.approx(8e9 / 64e12 * 1e3)
    assert r["bound"] == "l2" and r["t_lb_ms"] == max(t.values()) and r["frac"] == pytest.approx(r["t_lb_ms"] / 1.0)
    w["hbm_bytes"] = 6.5e9  # 1 ms of HBM traffic: now HBM binds
    assert bench.bounds(w, 2.0, peaks)["bound"] == "hbm"
    assert bench.bounds(w, 2.0, peaks)["frac"] == pytest.approx(0.5)


def test_lm_flop_count():
    assert bench.lm_flops_per_eval(29) == 92 * 29 + 300
    assert bench.lm_flops_per_step(29) == bench.lm_flops_per_eval(29) + 500
