"""SURVEY.md 8(f)1 on the CPU side: the K_i map of the oracle against exact rational arithmetic, the seeded noise
realisations, and the bias / variance bookkeeping of paper_1803_10045_b200/methods.py on maps with known statistics."""
from fractions import Fraction

import numpy as np

import kcs_inputs as ki
from oracle import Oracle


def test_ki_map_against_exact_fractions():
    """K_i = K1 k3 / (k2 + k3) for BASELINE's three tissue classes, in exact rational arithmetic; SURVEY 8(c) prints
    0.0329375 for grey matter."""
    regions = {"grey": ki.GREY, "white": ki.WHITE, "background": ki.BACKGROUND}
    th = np.array([regions[k] for k in regions]).T.reshape(4, 1, 1, 3)
    got = Oracle.ki_map(th).ravel()
    for q, k in enumerate(regions):
        K1, k2, k3, _ = (Fraction(str(v)) for v in regions[k])
        want = K1 * k3 / (k2 + k3)
        assert abs(got[q] - float(want)) <= 1e-16, (k, got[q], float(want))
    assert abs(got[0] - 0.0329375) <= 1e-16
    # k2 + k3 = 0 -> 0 (no uptake, no division); vB does not enter
    th0 = np.array([[0.3, 0.3], [0.0, 0.2], [0.0, 0.1], [0.1, 0.9]]).reshape(4, 1, 1, 2)
    np.testing.assert_allclose(Oracle.ki_map(th0).ravel(), [0.0, 0.1], rtol=1e-15)


def test_noise_realisations_are_seeded_and_independent():
    ybar = np.full((2, 3, 4, 5), 7.5)
    y = ki.noise_realisations(ybar, 11, 4)
    assert y.shape == (2, 12, 4, 5)
    assert np.array_equal(y[:, :3], ki.poisson(ybar, 11))            # realisation 0 is the single-run data
    assert np.array_equal(y, ki.noise_realisations(ybar, 11, 4))     # reproducible
    assert not np.array_equal(y[:, :3], y[:, 3:6])                   # realisations differ
    big = ki.noise_realisations(np.full((1, 1, 50, 50), 20.0), 3, 40)
    assert abs(big.mean() - 20.0) < 0.1 and abs(big.var() - 20.0) < 0.6   # Poisson: mean = variance


def test_region_statistics_of_known_maps():
    from paper_1803_10045_b200.methods import region_stats
    rng = np.random.default_rng(0)
    labels = np.zeros((1, 8, 8), dtype=np.int8)
    labels[0, :4] = 1
    labels[0, 4:] = 2
    mask = np.ones((8, 8), dtype=np.uint8)
    truth = np.where(labels == 1, 0.02, 0.04)
    n = 4000
    maps = truth[None] * (1.0 + np.where(labels == 1, 0.10, -0.05)[None]) + 0.1 * truth[None] * rng.standard_normal((n,) + truth.shape)
    st = region_stats(maps, labels, truth, mask)
    assert st["white"]["voxels"] == 32 and st["grey"]["voxels"] == 32
    assert abs(st["white"]["bias_pct"] - 10.0) < 0.3 and abs(st["grey"]["bias_pct"] + 5.0) < 0.3
    assert abs(st["white"]["cov_pct"] - 10.0) < 0.3 and abs(st["grey"]["cov_pct"] - 10.0) < 0.3
