"""Pins of the oracle's distance transform / soft-image synthesis (pipeline steps 1-2, section VII
l.342; reading DESIGN R17).  None of these checks re-types the oracle's own formula: they use the O(N^4) definition,
scipy's distance transform (a different algorithm), hand-computed values and the float64 evaluation of the harness."""
import numpy as np
import pytest

import scenes


def _walls(hard):
    h = hard.astype(bool).copy()
    h[0, :] = True
    h[:, 0] = True
    return h


def test_separable_form_equals_the_definition(oracle_mod):
    rng = np.random.default_rng(5)
    for n, p in ((8, 0.1), (16, 0.03), (24, 0.05), (24, 0.0), (16, 1.0)):
        hard = (rng.random((n, n)) < p).astype(np.uint8)
        d2, dist, soft = oracle_mod.soft_from_hard(hard)
        assert (d2 == oracle_mod.edt_brute(hard)).all(), (n, p)


def test_distance_against_scipy(oracle_mod):
    from scipy import ndimage
    rng = np.random.default_rng(6)
    images = [(rng.random((128, 128)) < 0.002).astype(np.uint8), scenes.get_config(4).hard, scenes.get_config(2).hard]
    for hard in images:
        d2, dist, _ = oracle_mod.soft_from_hard(hard)
        ref = ndimage.distance_transform_edt(~_walls(hard))
        assert np.abs(np.sqrt(d2.astype(np.float64)) - ref).max() < 1e-9
        assert np.abs(dist.astype(np.float64) - ref).max() <= 1e-5 * max(1.0, ref.max())      # float32 distance, north_star tolerance


def test_soft_values_by_hand(oracle_mod):
    # one hard pixel far from the walls: d = 0, 1, sqrt 2, 3, 4 -> 16 (1 + 4 / (d + 1)) = 80, 48, 42.51 -> 43, 32, 28.8 -> 29
    hard = np.zeros((64, 64), np.uint8)
    hard[40, 40] = 1
    d2, dist, soft = oracle_mod.soft_from_hard(hard, 4.0)
    assert soft[40, 40] == 80 and soft[40, 41] == 48 and soft[41, 41] == 43 and soft[40, 43] == 32 and soft[36, 40] == 29
    assert d2[41, 41] == 2 and d2[36, 40] == 16 and abs(dist[41, 41] - 2 ** 0.5) < 1e-6
    # walls count as hard: the pixel next to the wall column sees d = 1, the corner pixel (1, 1) too
    assert soft[20, 1] == 48 and soft[1, 1] == 48 and soft[0, 30] == 80
    # far from everything the multiplier tends to 1.0 = 16 and never drops below it
    assert soft.min() >= 16 and soft[20, 20] == int(np.rint(16 * (1 + 4 / (20 + 1))))
    # k = 0 switches the soft cost off
    assert (oracle_mod.soft_from_hard(hard, 0.0)[2] == 16).all()


def test_float32_evaluation_matches_the_float64_harness_away_from_ties(oracle_mod):
    sc = scenes.get_config(4)
    d2, dist, soft = oracle_mod.soft_from_hard(sc.hard, 4.0)
    ref = scenes.soft_from_hard(sc.hard, 4.0)                  # scipy distance, float64 formula
    diff = np.nonzero(soft != ref)
    exact = 16.0 * (1.0 + 4.0 / (np.sqrt(d2[diff].astype(np.float64)) + 1.0))
    assert len(diff[0]) < 1e-3 * soft.size
    assert (np.abs(exact - np.floor(exact) - 0.5) < 1e-5).all()      # only at rounding ties of rint
