"""Pins for the oracle's area / orientation penalty (orc_apply_lane, DESIGN R28).

The paper names the feature and gives no formula, so the definition is ours; the pins fix what any reading must satisfy (a
factor of 1.0 is the identity, the lane's own heading is free, the opposite heading pays the full factor) and what R28 adds
(linear in the angle, symmetric, evaluated at the pose's own pixel, heading measured from +x towards +y)."""
import numpy as np

import oracle

N, NT = 32, 32          # log2 5, 5: R = 4 satisfies N_theta >= 2 pi R


def make():
    return oracle.Oracle(5, 5, 4.0, (500, 100, 500, 500, 100, 500), (256,) * 6, 10, 0)


def volume(rng):
    return rng.integers(16, 256, size=(NT, N, N), dtype=np.uint8)


def test_factor_one_is_the_identity():
    o, rng = make(), np.random.default_rng(1)
    S = volume(rng)
    for pen in (np.full((N, N), 16, np.uint8), rng.integers(0, 17, size=(N, N), dtype=np.uint8)):      # values below 16 count as 16
        got = o.apply_lane(S.copy(), rng.integers(0, 256, size=(N, N), dtype=np.uint8), pen)
        assert (got == S).all()


def test_aligned_is_free_opposite_pays_the_factor_and_the_ramp_is_linear_and_symmetric():
    o, rng = make(), np.random.default_rng(2)
    S = volume(rng).astype(np.int64)
    for d0 in (0, 64, 40, 248):                                       # 40 and 248 are headings of planes 5 and 31
        for pen, mult in ((32, 2), (48, 3), (64, 4)):
            got = o.apply_lane(S.astype(np.uint8), np.full((N, N), d0, np.uint8), np.full((N, N), pen, np.uint8)).astype(np.int64)
            t0 = d0 * NT // 256                                       # the plane whose heading is exactly d0
            assert (got[t0] == S[t0]).all()
            assert (got[(t0 + NT // 2) % NT] == np.minimum(255, mult * S[(t0 + NT // 2) % NT])).all()       # exact product
            # a quarter turn away: half of the excess, on both sides
            for q in (NT // 4, -NT // 4):
                half = np.minimum(255, ((mult + 1) * S[(t0 + q) % NT] + 1) // 2)                              # (1 + mult) / 2, rounded half up
                assert (got[(t0 + q) % NT] == half).all()
            # symmetric in the angle and non-decreasing away from the lane direction; S itself differs per plane, so compare factors
            # on a constant volume
            flat = o.apply_lane(np.full((NT, N, N), 100, np.uint8), np.full((N, N), d0, np.uint8), np.full((N, N), pen, np.uint8))
            prof = flat[:, 3, 5].astype(int)
            for k in range(1, NT // 2 + 1):
                assert prof[(t0 + k) % NT] == prof[(t0 - k) % NT]
                assert prof[(t0 + k) % NT] >= prof[(t0 + k - 1) % NT]
            assert prof[t0] == 100 and prof[(t0 + NT // 2) % NT] == min(255, 100 * mult)


def test_monotone_in_the_factor_and_saturating():
    o, rng = make(), np.random.default_rng(3)
    S = volume(rng)
    d = rng.integers(0, 256, size=(N, N), dtype=np.uint8)
    prev = S.copy()
    for pen in (16, 20, 33, 64, 128, 255):
        got = o.apply_lane(S.copy(), d, np.full((N, N), pen, np.uint8))
        assert (got >= prev).all() and (got >= S).all()
        prev = got
    assert prev.max() == 255                                           # 255 * 255 / 16 saturates at 255, does not wrap


def test_the_penalty_is_read_at_the_pose_s_own_pixel():
    """Penalty only inside a non-square rectangle of pixels (rows = j, columns = i): exactly those poses change."""
    o = make()
    S = np.full((NT, N, N), 16, np.uint8)
    pen = np.full((N, N), 16, np.uint8)
    pen[5:9, 12:27] = 64                                               # j in 5..8, i in 12..26
    got = o.apply_lane(S.copy(), np.zeros((N, N), np.uint8), pen)
    changed = (got != S).any(axis=0)
    want = np.zeros((N, N), bool)
    want[5:9, 12:27] = True
    assert (changed == want).all()
    assert (got[NT // 2, 5:9, 12:27] == 64).all() and (got[0] == 16).all()


def test_driving_with_the_lane_is_free_and_against_it_costs_the_factor():
    """Free space, soft volume 1.0, lane direction +x (then +y) everywhere, factor 2.0.  A short straight drive that faces
    along the lane costs what it costs without the penalty; the same drive facing the other way costs exactly twice as much
    (edge weight = len * S >> 4 with S doubled, PAPER.md:338 'multiplied with the spatial length of each edge').  Fixes the
    angle convention: heading index Theta <-> angle 2 pi Theta / N_theta from +x towards +y."""
    o = make()
    fp = oracle.Footprint.box(1, 1)
    C, S0 = o.render(fp, np.zeros((N, N), np.uint8), np.full((N, N), 16, np.uint8), method="brute")
    assert (S0 == 16).all()
    len_sf = o.len_q[1]
    for lane_heading, with_, against, step in ((0, 0, NT // 2, (1, 0)), (64, NT // 4, 3 * NT // 4, (0, 1))):
        S1 = o.apply_lane(S0.copy(), np.full((N, N), lane_heading, np.uint8), np.full((N, N), 32, np.uint8))
        for theta, sign, factor in ((with_, 1, 1), (against, -1, 2)):
            start = (16, 16, theta)
            V0 = o.run(C, S0, start, 2)
            V1 = o.run(C, S1, start, 2)
            for d in (1, 2, 3):
                g = (theta, 16 + sign * d * step[1], 16 + sign * d * step[0])
                assert V0[g] == 100 + d * len_sf[theta]               # ct[SF] + d straight edges (axis heading: one cell each)
                if d == 1 or factor == 1:
                    assert V1[g] == 100 + factor * d * len_sf[theta], (lane_heading, theta, d)
                else:                                                  # further out a detour through cheaper headings may win
                    assert V0[g] < V1[g] <= 100 + factor * d * len_sf[theta], (lane_heading, theta, d)
