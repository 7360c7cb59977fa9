"""Pins of the oracle's goal search (section IX; reading DESIGN R20).  The checks are special cases
and properties that follow from "reward minus cost over a goal set", plus an independent numpy evaluation on window
slices; none calls the oracle's own loop to produce the expected value."""
import numpy as np
import pytest

import scenes

INF = 0xFFFFFFFF


@pytest.fixture(scope="module")
def solved(oracle_mod):
    sc = scenes.random_scene(6, 5, 5, 31, n_rects=8, n_cycles=4)
    o = oracle_mod.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct, sc.dir_mult, sc.cost_one_log2, sc.flags, threads=0)
    fp = oracle_mod.Footprint(sc.mask, sc.ou, sc.ov)
    Cv, Sv = o.render(fp, sc.hard, sc.soft)
    V = o.run(Cv, Sv, sc.start, sc.n_cycles)
    return sc, o, Cv, V


def reached_goals(V, n, rng, margin=6):
    t, j, i = np.nonzero(V != INF)
    ok = (i >= margin) & (i < n - margin) & (j >= margin) & (j < n - margin)
    pick = rng.choice(np.nonzero(ok)[0], size=12, replace=False)
    return [(int(i[k]), int(j[k]), int(t[k])) for k in pick]


def test_radius_zero_is_the_explicit_goal(solved):
    sc, o, Cv, V = solved
    for g in reached_goals(V, sc.n, np.random.default_rng(1)):
        cell, gi, score = o.goal_search(V, [g], 0, 1000, 1000)
        assert cell == g and gi == 0 and score == int(V[g[2], g[1], g[0]])


def test_large_weights_keep_the_ideal_pose_and_zero_weights_take_the_cheapest(solved):
    sc, o, Cv, V = solved
    nt = sc.nt
    for g in reached_goals(V, sc.n, np.random.default_rng(2)):
        cell, _, score = o.goal_search(V, [g], 3, 1 << 19, 1 << 19)
        assert cell == g                                                     # no alignment is worth 2^19 cost units here
        cell, _, score = o.goal_search(V, [g], 3, 0, 0)
        ts = [(g[2] + dt) % nt for dt in range(-3, 4)]
        win = V[ts][:, g[1] - 3:g[1] + 4, g[0] - 3:g[0] + 4].astype(np.int64)
        dj, di = np.mgrid[-3:4, -3:4]
        win[:, (di * di + dj * dj) > 9] = INF                                # the goal set is a disc in (i, j)
        assert score == win.min() and int(V[cell[2], cell[1], cell[0]]) == score


def test_score_is_cost_plus_quadratic_penalty_and_never_worse_than_the_ideal_pose(solved):
    sc, o, Cv, V = solved
    rng = np.random.default_rng(3)
    for g in reached_goals(V, sc.n, rng):
        W, w = int(rng.integers(1, 5000)), int(rng.integers(1, 5000))
        cell, _, score = o.goal_search(V, [g], 4, W, w)
        di, dj = cell[0] - g[0], cell[1] - g[1]
        dt = (cell[2] - g[2] + sc.nt // 2) % sc.nt - sc.nt // 2
        assert di * di + dj * dj <= 16 and abs(dt) <= 4
        assert score == int(V[cell[2], cell[1], cell[0]]) + W * (di * di + dj * dj) + w * dt * dt
        assert score <= int(V[g[2], g[1], g[0]])                              # the ideal pose itself is in the set
        # monotone in the radius: a larger goal set can only improve the criterion
        assert o.goal_search(V, [g], 5, W, w)[2] <= score <= o.goal_search(V, [g], 2, W, w)[2]


def test_several_ideal_goals_and_empty_sets(solved, oracle_mod):
    sc, o, Cv, V = solved
    goals = reached_goals(V, sc.n, np.random.default_rng(4))
    single = [o.goal_search(V, [g], 2, 300, 700) for g in goals]
    cell, gi, score = o.goal_search(V, goals, 2, 300, 700)
    assert score == min(s[2] for s in single)
    first = min(k for k, s in enumerate(single) if s[2] == score)              # ties go to the earlier goal
    assert gi == first and cell == single[first][0]
    # a goal set entirely inside an obstacle (or unreached) is empty: code -5, like an unreached explicit goal
    t, j, i = np.nonzero(Cv != 0)
    deep = [(int(i[k]), int(j[k]), int(t[k])) for k in range(len(i)) if V[t[k], max(j[k] - 1, 0):j[k] + 2, max(i[k] - 1, 0):i[k] + 2].min() == INF
            and 2 < i[k] < sc.n - 2 and 2 < j[k] < sc.n - 2 and (V[[(t[k] - 1) % sc.nt, (t[k] + 1) % sc.nt]][:, j[k] - 1:j[k] + 2, i[k] - 1:i[k] + 2] == INF).all()]
    assert deep
    with pytest.raises(oracle_mod.OracleError) as e:
        o.goal_search(V, [deep[0]], 1, 1, 1)
    assert e.value.code == -5
    # the window is clipped at the grid border (no spatial wrap)
    cell, _, _ = o.goal_search(V, [sc.start], 3, 0, 0)
    assert 0 <= cell[0] < sc.n and 0 <= cell[1] < sc.n
