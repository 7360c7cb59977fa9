"""Pins for the oracle's maneuver sweeps, N-turn driver and Dijkstra."""
import numpy as np
import pytest

import oracle
import scenes
from helpers import INF, closed_form_sweep, pm26_reach, random_volume


def make(sc, **kw):
    return oracle.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct, sc.dir_mult, sc.cost_one_log2, sc.flags, **kw)


def rendered(sc, o=None):
    o = o or make(sc)
    fp = oracle.Footprint(sc.mask, sc.ou, sc.ov)
    C, S = o.render(fp, sc.hard, sc.soft, method="brute")
    return o, C, S


@pytest.mark.parametrize("soft", [False, True])
def test_single_sweep_equals_closed_form(soft):
    """One maneuver kernel (Insert 5 l.946-949) == the closed form over < one lap of sources,
    on random values, random blocked cells and random soft multipliers, for all six maneuvers; this also
    shows that two laps of a cyclic curve are enough (l.356) and that saturation behaves."""
    rng = np.random.default_rng(5)
    o = oracle.Oracle(3, 4, 2, (700, 0, 900, 650, 300, 1 << 20), (256, 256, 512, 256, 300, 256))
    for trial in range(3):
        V, C, S = random_volume(rng, o.shape, vmax=[5000, 1 << 29, (1 << 30) - 1][trial])
        S = S if soft else None
        for m in range(6):
            got = V.copy()
            o.sweep(m, got, C, S)
            want = closed_form_sweep(o, m, V, C, S)
            assert (got == want).all(), (m, trial)
            assert (got[C != 0] == INF).all()


@pytest.mark.parametrize("seed,soft,rev", [(1, False, 256), (2, True, 512), (3, True, 256)])
def test_fixpoint_equals_star_dijkstra(seed, soft, rev):
    """Iterating maneuver cycles converges to the exact shortest-path values of the Star graph built from the
    edge maps (25)-(31); cycles decrease monotonically towards it."""
    sc = scenes.random_scene(5, 5, 4, seed, soft=soft, reverse_mult=rev)
    o, C, S = rendered(sc)
    D = o.dijkstra(C, S, sc.start, "star")
    V = o.run(C, S, sc.start, 1)
    assert V[sc.start[2], sc.start[1], sc.start[0]] == 0
    for k in range(40):
        assert (V >= D).all()
        V2 = V.copy()
        o.cycles(V2, C, S, 1)
        assert (V2 <= V).all()
        if (V2 == V).all():
            break
        V = V2
    assert k < 39
    assert (V == D).all()
    assert (V[C != 0] == INF).all()
    assert (V != INF).sum() > 0.2 * (C == 0).sum()


def test_compact_graph_dijkstra_matches_when_weights_conform():
    """with conforming costs the 3-vertex / 10-edge Compact graph has the same values."""
    sc = scenes.random_scene(5, 5, 4, 11, soft=True, ct=(4096, 0, 5000, 5000, 0, 4096))
    o, C, S = rendered(sc)
    Dc = o.dijkstra(C, S, sc.start, "compact")
    Ds = o.dijkstra(C, S, sc.start, "star")
    V = o.run(C, S, sc.start, 12)
    assert (Dc == Ds).all() and (V == Ds).all()
    sc2 = scenes.random_scene(5, 5, 4, 11)                       # COUNTING weights do not conform
    with pytest.raises(oracle.OracleError):
        make(sc2).dijkstra(C, None, sc.start, "compact")


def test_forward_only_is_a_dubins_car():
    sc = scenes.random_scene(5, 5, 4, 21, flags=oracle.FLAG_FORWARD_ONLY)
    o, C, S = rendered(sc)
    V = o.run(C, S, sc.start, 10)
    assert (V == o.dijkstra(C, S, sc.start, "star")).all()
    full = make(scenes.random_scene(5, 5, 4, 21))
    assert (full.run(C, S, sc.start, 10) <= V).all()


def test_n_cycles_cover_all_n_maneuver_plans():
    """N_T cycles evaluate all N_T-maneuver plans.  W_n = best cost over plans of <= n maneuvers,
    by an independent layered (Jacobi) DP built on the closed form; then V_n <= W_n and V_n >= V_inf."""
    sc = scenes.random_scene(3, 4, 2, 4, n_rects=2, max_side=2, vehicle=(1, 1))
    o, C, S = rendered(sc)
    D = o.dijkstra(C, S, sc.start, "star")
    W = np.full(o.shape, INF, np.uint32)
    W[sc.start[2], sc.start[1], sc.start[0]] = 0
    for ncyc in range(1, 4):
        W = np.minimum.reduce([closed_form_sweep(o, m, W, C, S) for m in range(6)])
        V = o.run(C, S, sc.start, ncyc)
        assert (V <= W).all()
        assert (V >= D).all()
    assert (W != INF).sum() > 20


def test_free_space_closed_forms():
    """Straight ahead k cells costs ct + k * length; k steps along an arc cost ct + k * 2 pi R / N_theta
    (Lemma 4/5 l.779-785: the edge lengths add up to the exact segment / arc length)."""
    n, nt, R = 64, 64, 8
    ct = (9000, 8000, 9100, 9200, 8100, 9300)
    o = oracle.Oracle(6, 6, R, ct)
    fp = oracle.Footprint(np.ones((1, 1), np.uint8), 0.0, 0.0)
    C, _ = o.render(fp, np.zeros((n, n), np.uint8))
    assert C[:, 0, :].all() and C[:, :, 0].all()                 # the wall of PAPER.md:226
    assert C[:, 1:-1, 1:-1].sum() == 0                           # (half-cell poses next to the seam touch it)
    lq = o.len_q
    for t0 in (0, 5, 8, 13, 16, 29, 40, 63):
        start = (30, 33, t0)
        V = o.run(C, None, start, 1)
        for m in range(6):
            p, acc = start, ct[m]
            for k in range(1, 6):
                acc += int(lq[m, p[2]])
                p = o.edge(m, *p)
                assert V[p[2], p[1], p[0]] == acc, (t0, m, k)
    # exact geometry: 16 LF steps from heading 0 is a quarter circle of radius R (eq (1) with q = +1)
    p = (30, 33, 0)
    for _ in range(16):
        p = o.edge(oracle.LF, *p)
    psi2 = o.psi2
    x = p[0] + psi2[p[2]] / 2 - 30
    y = p[1] + psi2[(p[2] + 16) % 64] / 2 - 33
    assert p[2] == 16 and abs(x - R) <= 0.5 and abs(y - R) <= 0.5


def test_piano_mover_relaxation_bounds():
    """every maneuver edge moves each of (i, j, Theta) by at most one cell (l.269), so the
    nonholonomic reach set is inside the 26-neighbour Piano-mover flood fill of the same collision volume
    and V_inf >= ct + steps_PM26 * (cheapest edge)."""
    sc = scenes.random_scene(5, 5, 4, 9, n_rects=8)
    o, C, S = rendered(sc)
    V = o.dijkstra(C, None, sc.start, "star")
    steps = pm26_reach(C, sc.start)
    reached = V != INF
    assert (steps[reached] >= 0).all()
    wmin = int(o.len_q.min())
    lower = np.where(steps > 0, min(sc.ct) + steps * wmin, 0)
    assert (V[reached] >= lower[reached]).all()
    assert reached.sum() > 1000


def test_seam_is_closed():
    """a one-cell wall at i = 0 and j = 0 makes the toroidal addressing safe."""
    sc = scenes.random_scene(5, 5, 4, 2, n_rects=0, vehicle=(1, 1))
    o = make(sc)
    fp = oracle.Footprint(sc.mask, sc.ou, sc.ov)
    C, _ = o.render(fp, sc.hard, None, method="brute")
    V = o.run(C, None, (3, 16, 16), 8)                           # 3 cells from the border, heading -x
    assert (V[:, 0, :] == INF).all() and (V[:, :, 0] == INF).all()
    assert (V[C != 0] == INF).all()
    assert (V != INF).sum() > 0.95 * (C == 0).sum()               # nearly everything else is reachable in free space
    with pytest.raises(oracle.OracleError) as e:
        o.run(C, None, (0, 5, 5), 1)
    assert e.value.code == -4
