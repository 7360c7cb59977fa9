"""Pins of the start state with a maneuver in progress (section XII; reading DESIGN R26)."""
import numpy as np
import pytest

import scenes

INF = 0xFFFFFFFF


@pytest.fixture(scope="module")
def world(oracle_mod):
    sc = scenes.random_scene(5, 5, 4, 41, n_rects=5, n_cycles=3, soft=True, reverse_mult=384)
    o = oracle_mod.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct, sc.dir_mult, sc.cost_one_log2, sc.flags, threads=0)
    fp = oracle_mod.Footprint(sc.mask, sc.ou, sc.ov)
    Cv, Sv = o.render(fp, sc.hard, sc.soft)
    return sc, o, Cv, Sv


def test_fix_point_equals_star_dijkstra_with_the_maneuver_vertex_as_a_source(world):
    """'No transition cost to start with that maneuver' = the Star vertex (start, m0) is a source besides T(start)."""
    sc, o, Cv, Sv = world
    for m0 in range(6):
        V = o.run_from(Cv, Sv, sc.start, m0, 1)
        for _ in range(12):
            W = V.copy()
            o.cycles(V, Cv, Sv, 1)
            if (V == W).all():
                break
        assert (V == o.dijkstra(Cv, Sv, sc.start, "star", m0)).all(), m0


def test_first_maneuver_is_free_and_everything_else_unchanged(world, oracle_mod):
    sc, o, Cv, Sv = world
    plain = o.run(Cv, Sv, sc.start, 3)
    assert (o.run_from(Cv, Sv, sc.start, -1, 3) == plain).all()
    for m0 in range(6):
        V = o.run_from(Cv, Sv, sc.start, m0, 3)
        assert (V <= plain).all() and V[sc.start[2], sc.start[1], sc.start[0]] == 0
        # one edge ahead on the curve of m0: exactly the edge weight at the start vertex, no c_t (if that vertex is free)
        i2, j2, t2 = o.edge(m0, *sc.start)
        if not Cv[t2, j2, i2]:
            w = (int(o.len_q[m0][sc.start[2]]) * int(Sv[sc.start[2], sc.start[1], sc.start[0]])) >> 4
            assert V[t2, j2, i2] == min(w, int(plain[t2, j2, i2]))
        # at the fix-point the gain is at most the transition cost of m0 (enter m0 from T(start) instead)
        D0, Dm = o.dijkstra(Cv, Sv, sc.start, "star"), o.dijkstra(Cv, Sv, sc.start, "star", m0)
        both = (D0 != INF)
        assert ((Dm != INF) == both).all() and (Dm <= D0).all()
        assert ((D0[both].astype(np.int64) - Dm[both].astype(np.int64)) <= sc.ct[m0]).all()


def test_plan_accounts_for_the_free_first_maneuver(world, oracle_mod):
    sc, o, Cv, Sv = world
    rng = np.random.default_rng(3)
    for m0 in (0, 1, 3, 4):
        V = o.run_from(Cv, Sv, sc.start, m0, 8)
        t, j, i = np.nonzero(V != INF)
        for k in rng.integers(len(t), size=25):
            goal = (int(i[k]), int(j[k]), int(t[k]))
            plan, cost = o.backtrack_from(V, Cv, Sv, sc.start, m0, goal)
            assert plan[0][:3] == goal and plan[-1] == tuple(sc.start) + (-1,)
            assert cost == int(V[goal[2], goal[1], goal[0]])          # converged volume: the plan's cost is the vertex value
