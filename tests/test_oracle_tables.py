"""Pins for the oracle's tables, curve maps and edge maps.

Nothing here re-types the oracle's formulas: the checks are the invariants and bounds the paper
states about them (Lemma 4/5 l.779-785) and
the numbers of its worked example (tests/golden/paper_constants.txt).
"""
import math
import os

import numpy as np
import pytest

import oracle

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as f:
    for line in f:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = float(line[1])

# (log2_n, log2_nt, R) of the five BASELINE.json configs
CONFIG_GRIDS = [(6, 6, 8), (8, 8, 30), (9, 9, 12), (9, 9, 40), (10, 9, 50)]


def make(log2_n, log2_nt, R, **kw):
    return oracle.Oracle(log2_n, log2_nt, R, (int(R * 1024),) * 6, **kw)


@pytest.mark.parametrize("log2_n,log2_nt,R", CONFIG_GRIDS + [(5, 5, 4), (4, 6, 7.3)])
def test_turn_tables_identities_and_snap_error(log2_n, log2_nt, R):
    o = make(log2_n, log2_nt, R)
    nt, q = o.nt, o.nt // 4
    beta, psi2 = o.beta.astype(np.int64), o.psi2.astype(np.int64)
    th = 2 * np.pi * np.arange(nt) / nt
    # Psi in {0, 1/2};  Psi_2 = Psi_0 and Psi_3 = Psi_1
    assert set(np.unique(psi2)) <= {0, 1}
    assert (np.roll(psi2, -2 * q) == psi2).all()
    assert (np.roll(psi2, -3 * q) == np.roll(psi2, -q)).all()
    # snap error of the rounded turn curve <= 1/4 cell (Lemma 4 l.779)
    err = np.abs(beta + psi2 / 2.0 - R * np.sin(th))
    assert err.max() <= GOLD["turn_snap_error"] + 1e-9
    # successive planes shift by at most one pixel when N_theta >= 2 pi R
    assert np.abs(np.roll(beta, -1) - beta).max() <= 1
    # the four quarter-period references are sin, cos, -sin, -cos
    for k, ref in enumerate((np.sin(th), np.cos(th), -np.sin(th), -np.cos(th))):
        bk = np.roll(beta, -k * q) + np.roll(psi2, -k * q) / 2.0
        assert np.abs(bk - R * ref).max() <= 0.25 + 1e-9


@pytest.mark.parametrize("log2_n,log2_nt,R", CONFIG_GRIDS + [(5, 5, 4)])
def test_straight_tables(log2_n, log2_nt, R):
    o = make(log2_n, log2_nt, R)
    n, nt = o.n, o.nt
    th = 2 * np.pi * np.arange(nt) / nt
    I, J, K, B = o.I, o.J, o.K, o.B
    t, c, s = np.tan(th), np.cos(th), np.sin(th)
    # eq (19): I = 0 iff |tan| <= 1 (away from the four exact diagonals, where FP tan is off by an ulp)
    diag = (np.arange(nt) % (nt // 4)) == nt // 8
    assert ((I == 0) == (np.abs(t) <= 1))[~diag].all()
    assert (I[diag] == 0).all() and (np.abs(np.abs(K[diag]) - 1.0) == 0).all()
    # eq (20) and the 1/2 cell rounding bound of eq (22) (Lemma 5 l.783)
    Kref = np.where(I == 0, t, 1.0 / np.where(t == 0, 1, t))
    assert np.abs(K - Kref)[~diag].max() < 1e-12
    y = np.arange(n)[None, :]
    assert np.abs(B - y * K[:, None]).max() <= GOLD["straight_snap_error"] + 1e-9
    assert np.abs(np.diff(B, axis=1)).max() <= 1
    # eq (24): forward direction
    Jref = np.where(I == 0, np.sign(c), np.sign(s))
    assert (J == Jref).all()
    # edge lengths PAPER.md:334: turn 2 pi R / N_theta, straight 1/|cos| or 1/|sin|, in 1/1024 cell
    lq = o.len_q.astype(np.float64) / 1024.0
    ls = np.where(I == 0, 1 / np.abs(c), 1 / np.abs(np.where(s == 0, 1, s)))
    for m in (oracle.SF, oracle.SB):
        assert np.abs(lq[m] - ls).max() <= 0.5 / 1024 + 1e-12
    for m in (oracle.LF, oracle.LB, oracle.RF, oracle.RB):
        assert np.abs(lq[m] - 2 * np.pi * R / nt).max() <= 0.5 / 1024 + 1e-12
    assert lq[oracle.SF].min() >= 1.0 and lq[oracle.SF].max() <= math.sqrt(2) + 1e-3


def test_worked_example_angular_resolution():
    """d_x = 0.125 m, R = 10 m -> N_theta >= 503, so 512 passes and 256 is refused."""
    R_cells = GOLD["example_R_m"] / GOLD["example_dx_m"]
    assert math.ceil(2 * math.pi * R_cells) == GOLD["example_ntheta_min"]
    assert math.degrees(GOLD["example_dx_m"] / GOLD["example_dc_m"]) == pytest.approx(GOLD["example_dtheta_deg"], abs=0.05)
    make(10, 9, R_cells)                                   # 512 angles: accepted
    with pytest.raises(oracle.OracleError) as e:
        make(10, 8, R_cells)                               # 256 angles: N_theta < 2 pi R
    assert e.value.code == 2


def _all_cells(o, m):
    n, nt = o.n, o.nt
    turn = m not in (oracle.SF, oracle.SB)
    out = {}
    for c1 in range(n if turn else nt):
        for c0 in range(n):
            for k in range(nt if turn else n):
                out[(c0, c1, k)] = o.curve_cell(m, c0, c1, k)
    return out


@pytest.mark.parametrize("log2_n,log2_nt,R", [(4, 5, 4), (3, 5, 5)])
def test_curve_maps_are_bijections_and_edges_follow_curves(log2_n, log2_nt, R):
    """the curves of one maneuver are a disjoint cover of the volume;
    l.306, l.320: an edge map = inverse curve map, one step along the sweep coordinate, curve map."""
    o = make(log2_n, log2_nt, R)
    n, nt = o.n, o.nt
    J = o.J
    for m in range(6):
        cells = _all_cells(o, m)
        assert len(set(cells.values())) == n * n * nt == len(cells)
        turn = m not in (oracle.SF, oracle.SB)
        for (c0, c1, k), (i, j, t) in cells.items():
            if turn:
                step = 1 if m in (oracle.LF, oracle.RB) else -1      # Theta up for LF, RB (eq 25, 28)
                nxt = cells[(c0, c1, (k + step) % nt)]
            else:
                step = 1 if (m == oracle.SF) == (J[c1] > 0) else -1
                nxt = cells[(c0, c1, (k + step) % n)]
            assert o.edge(m, i, j, t) == nxt
    # forward and backward versions of a maneuver retrace each other
    rng = np.random.default_rng(0)
    for _ in range(300):
        p = (int(rng.integers(n)), int(rng.integers(n)), int(rng.integers(nt)))
        for a, b in ((oracle.LF, oracle.LB), (oracle.RF, oracle.RB), (oracle.SF, oracle.SB)):
            assert o.edge(b, *o.edge(a, *p)) == p
            assert o.edge(a, *o.edge(b, *p)) == p
    # a full turn closes after N_theta steps; every maneuver edge moves each coordinate by <= 1 (l.269)
    for m in (oracle.LF, oracle.RF):
        p = q = (3, 5, 7)
        for _ in range(nt):
            q2 = o.edge(m, *q)
            d = [min((a - b) % s, (b - a) % s) for a, b, s in zip(q2, q, (n, n, nt))]
            assert max(d) <= 1
            q = q2
        assert q == p


def test_turn_directions_match_the_continuum_model():
    """PAPER.md:92 dynamics v(cos, sin, k): a left-forward step increases theta and moves along the heading;
    eq (1): left turns have their centre on the left."""
    o = make(7, 8, 20)
    n, nt = o.n, o.nt
    psi2 = o.psi2
    def pos(p):
        return np.array([p[0] + psi2[p[2]] / 2.0, p[1] + psi2[(p[2] + nt // 4) % nt] / 2.0])
    for m, dth, sgn in ((oracle.LF, 1, 1), (oracle.LB, -1, -1), (oracle.RF, -1, 1), (oracle.RB, 1, -1),
                        (oracle.SF, 0, 1), (oracle.SB, 0, -1)):
        for t0 in range(0, nt, 5):
            p = (60, 64, t0)
            q = p
            for _ in range(6):
                q = o.edge(m, *q)
            assert (q[2] - p[2]) % nt == (6 * dth) % nt
            d = pos(q) - pos(p)
            th = 2 * np.pi * (t0 + 3 * dth) / nt
            heading = np.array([np.cos(th), np.sin(th)])
            # six steps of length ~2 pi R / N_theta (turn) or 1/max(|cos|,|sin|) (straight) along +-heading
            assert sgn * float(d @ heading) > 1.5
            assert abs(float(d @ np.array([-heading[1], heading[0]]))) < 1.6


def test_graph_sizes_of_table_1():
    """PAPER.md:427 and Table 1 l.436-437: the Star graph has k_V = 7 vertices and k_E = 18 edges per configuration X,
    the Compact graph 3 and 10 (tests/golden/paper_constants.txt).  Counted on the oracle's own Dijkstra at an interior
    cell of free space: the vertices of X it settles and the edges it relaxes out of them."""
    ct = (4096, 0, 5000, 5000, 0, 4096)                          # conforming weights, so that both graphs apply
    o = oracle.Oracle(5, 5, 4, ct)
    fp = oracle.Footprint(np.ones((1, 1), np.uint8), 0.0, 0.0)
    C, _ = o.render(fp, np.zeros((32, 32), np.uint8))
    for cell in ((16, 16, 3), (9, 20, 30)):
        assert o.graph_size_at(C, None, (12, 12, 0), cell, "star") == (GOLD["kV_star"], GOLD["kE_star"])
        assert o.graph_size_at(C, None, (12, 12, 0), cell, "compact") == (GOLD["kV_compact"], GOLD["kE_compact"])
    # the Piano-mover's graph of the comparison: one vertex, six neighbours (tests/helpers.py uses its 26-neighbour relaxation)
    assert (GOLD["kV_piano"], GOLD["kE_piano"]) == (1, 6)
    # forward only: the three reverse maneuver vertices and their edges disappear (Dubins car)
    of = oracle.Oracle(5, 5, 4, ct, flags=oracle.FLAG_FORWARD_ONLY)
    assert of.graph_size_at(C, None, (12, 12, 0), (16, 16, 3), "star") == (4, 9)
