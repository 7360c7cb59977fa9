"""Pins for the oracle's back-tracking (eq (32))."""
import numpy as np
import pytest

import oracle
import scenes
from helpers import INF, LIMIT


def check_plan(o, V, C, S, start, goal, plan, cost):
    """A plan is a chain of whole-curve segments: walking FORWARD along maneuver m from waypoint k+1 reaches
    waypoint k over free cells; ct + the edge weights (charged at their sources) add up to the reported cost."""
    assert plan[0][:3] == tuple(goal) and plan[-1][:3] == tuple(start) and plan[-1][3] == -1
    lenq = o.len_q
    total = 0
    for (gi, gj, gt, m), (si, sj, st, _) in zip(plan[:-1], plan[1:]):
        assert 0 <= m < 6
        p, seg = (si, sj, st), 0
        for _ in range(max(o.n, o.nt)):
            assert C[p[2], p[1], p[0]] == 0
            sv = 16 if S is None else int(S[p[2], p[1], p[0]])
            seg += (int(lenq[m, p[2]]) * sv) >> 4
            p = o.edge(m, *p)
            if p == (gi, gj, gt):
                break
        else:
            raise AssertionError("waypoints are not on one curve of the stated maneuver")
        assert C[gt, gj, gi] == 0
        total += o.ct[m] + seg
    assert total == cost < LIMIT
    return total


@pytest.mark.parametrize("seed,soft,rev", [(1, False, 256), (5, True, 512), (8, True, 256)])
def test_plans_are_valid_and_optimal_when_converged(seed, soft, rev):
    sc = scenes.random_scene(5, 5, 4, seed, soft=soft, reverse_mult=rev)
    o = oracle.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct, sc.dir_mult)
    fp = oracle.Footprint(sc.mask, sc.ou, sc.ov)
    C, S = o.render(fp, sc.hard, sc.soft)
    Vinf = o.dijkstra(C, S, sc.start, "star")
    rng = np.random.default_rng(seed)
    tj, jj, ij = np.nonzero(Vinf != INF)
    picks = rng.integers(len(tj), size=25)
    for ncyc, converged in ((2, False), (12, True)):
        V = o.run(C, S, sc.start, ncyc)
        if converged:
            assert (V == Vinf).all()
        for k in picks:
            goal = (int(ij[k]), int(jj[k]), int(tj[k]))
            vg = int(V[goal[2], goal[1], goal[0]])
            try:
                plan, cost = o.backtrack(V, C, S, sc.start, goal)
            except oracle.OracleError as e:
                # only a goal whose value is still infinite may be reported unreached; even then one more
                # reverse Bellman step can find it (the minimum may be below V[goal] before convergence)
                assert e.code == -5 and vg == INF
                continue
            check_plan(o, V, C, S, sc.start, goal, plan, cost)
            # PAPER.md:382 "the smallest value should be exactly the value of the current vertex"
            assert cost <= vg
            assert cost >= int(Vinf[goal[2], goal[1], goal[0]])
            if converged:
                assert cost == vg


def test_degenerate_goals():
    sc = scenes.random_scene(5, 5, 4, 3)
    o = oracle.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct)
    fp = oracle.Footprint(sc.mask, sc.ou, sc.ov)
    C, S = o.render(fp, sc.hard, None)
    V = o.run(C, S, sc.start, 4)
    plan, cost = o.backtrack(V, C, S, sc.start, sc.start)
    assert plan == [tuple(sc.start) + (-1,)] and cost == 0
    with pytest.raises(oracle.OracleError) as e:
        o.backtrack(V, C, S, sc.start, (0, 5, 5))           # a wall cell
    assert e.value.code == -5
    # one straight segment ahead of the start: a two-waypoint plan with the closed-form cost
    p, acc = tuple(sc.start), sc.ct[oracle.SF]
    for _ in range(3):
        acc += int(o.len_q[oracle.SF, p[2]])
        p = o.edge(oracle.SF, *p)
        if C[p[2], p[1], p[0]]:
            pytest.skip("start faces an obstacle")
    plan, cost = o.backtrack(V, C, S, sc.start, p)
    assert cost == acc and plan == [p + (oracle.SF,), tuple(sc.start) + (-1,)]
    with pytest.raises(oracle.OracleError) as e:
        o.backtrack(V, C, S, sc.start, sc.goal, cap=1)
    assert e.value.code in (-6, -5)
