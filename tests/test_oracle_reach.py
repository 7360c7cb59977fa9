"""Pins of the oracle's reachability ("bit-vector") planner, appendix C."""
import numpy as np
import pytest

import scenes

INF = 0xFFFFFFFF


@pytest.fixture(scope="module")
def world(oracle_mod):
    sc = scenes.random_scene(5, 5, 4, 61, n_rects=5)
    o = oracle_mod.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct, sc.dir_mult, sc.cost_one_log2, sc.flags, threads=0)
    fp = oracle_mod.Footprint(sc.mask, sc.ou, sc.ov)
    Cv, _ = o.render(fp, sc.hard, None)
    return sc, o, Cv


def test_level_of_a_vertex_is_the_fewest_maneuvers_of_the_star_graph(world, oracle_mod):
    """'Edge weights are zero for maneuver edges and one for transition edges' (l.871): the level volumes are the balls of
    that metric.  Checked with the Star Dijkstra under weights where one maneuver costs 2^20 and one edge costs 1 (fewer
    than 2^20 edges fit a path of a 32^3 grid), so cost >> 20 = number of maneuvers."""
    sc, o, Cv = world
    od = oracle_mod.Oracle(sc.log2_n, sc.log2_nt, sc.R, (1 << 20,) * 6, (256,) * 6, 0, sc.flags, threads=0)
    assert (od.len_q == 1).all()
    D = od.dijkstra(Cv, None, sc.start, "star")
    K = o.reach_run(Cv, sc.start, 40)
    fin = D != INF
    assert ((K != 255) == fin).all()                       # 40 levels are a fix-point here
    assert (K[fin] == (D[fin] >> 20)).all()
    assert K[sc.start[2], sc.start[1], sc.start[0]] == 0 and (K[Cv != 0] == 255).all()


def test_levels_are_nested_and_a_prefix_of_the_fix_point(world):
    sc, o, Cv = world
    full = o.reach_run(Cv, sc.start, 40)
    for n_levels in (0, 1, 2, 3, 5):
        K = o.reach_run(Cv, sc.start, n_levels)
        assert (K[full <= n_levels] == full[full <= n_levels]).all() and (K[full > n_levels] == 255).all()
    assert (o.reach_run(Cv, sc.start, 0) != 255).sum() == 1


def test_kernel_style_sweeps_reach_at_least_the_same_level(world):
    """N cycles of the in-place value sweeps evaluate every plan of <= N maneuvers: whatever the Jacobi levels
    reach with N maneuvers is finite in the value volume after N cycles."""
    sc, o, Cv = world
    for n in (1, 2, 3):
        V = o.run(Cv, None, sc.start, n)
        K = o.reach_run(Cv, sc.start, n)
        assert (V[K != 255] != INF).all()


def test_plans_have_exactly_level_many_maneuvers_and_follow_free_curves(world):
    sc, o, Cv = world
    K = o.reach_run(Cv, sc.start, 40)
    rng = np.random.default_rng(5)
    t, j, i = np.nonzero((K != 255) & (K > 0))
    for k in rng.integers(len(t), size=40):
        goal = (int(i[k]), int(j[k]), int(t[k]))
        plan, cost = o.reach_backtrack(K, Cv, sc.start, goal)
        assert cost == K[goal[2], goal[1], goal[0]] == len(plan) - 1
        assert plan[0][:3] == goal and plan[-1] == tuple(sc.start) + (-1,)
        for a, b in zip(plan[:-1], plan[1:]):
            # b -> a along maneuver a[3]: walk the edge map forward from b, every vertex free, until a
            m, cur = a[3], b[:3]
            for _ in range(max(sc.n, sc.nt)):
                cur = o.edge(m, *cur)
                assert not Cv[cur[2], cur[1], cur[0]]
                if cur == a[:3]:
                    break
            assert cur == a[:3]
            assert K[b[2], b[1], b[0]] == K[a[2], a[1], a[0]] - 1
