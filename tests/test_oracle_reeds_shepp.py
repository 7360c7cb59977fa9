"""Pin of the oracle against the free-space closed forms of the Dubins and Reeds-Shepp vehicles.

PAPER.md:104 (Theorem 1), l.809 (Theorem 6), l.815 (Theorem 7): without obstacles and with maneuver-counting
transition costs, the graph's reachable sets are at most 4 grid cells larger (same angle) and at most
7 + pi d / N_theta cells (4 angular cells) smaller than the continuum vehicle's.  The continuum side is
tests/closed_forms.py (written from the geometry, pinned in test_closed_forms_* below); the graph side is the oracle's
exact fix-point (Star Dijkstra; tests/test_oracle_sweeps.py shows that the maneuver cycles converge to it).  A global
mistake of the graph -- turn radius, handedness against gear, the heading convention, a transition cost lost or doubled
at a gear reversal, straight lengths on the skewed lines -- moves V_inf by whole transition costs or by tens of per
cent of the path length and fails one of the three checks.
"""
import numpy as np
import pytest

import oracle
from closed_forms import dubins, endpoint, mod2pi, reeds_shepp

ONE_LOG2 = 10
ONE = 1 << ONE_LOG2
INF = 0xFFFFFFFF


# ---------------------------------------------------------------------------------------------------------------
# the closed forms themselves
# ---------------------------------------------------------------------------------------------------------------
def _seen_after(prim, s, x, y, phi):
    """The goal (x, y, phi) as seen from the pose reached by driving primitive `prim` for the signed length s."""
    px, py, pth = endpoint(prim, [np.full_like(x, s)])
    dx, dy = x - px, y - py
    c, sn = np.cos(pth), np.sin(pth)
    return dx * c + dy * sn, -dx * sn + dy * c, mod2pi(phi - pth)


def test_closed_forms_known_values_and_symmetries():
    R = 3.0
    assert reeds_shepp(7.5, 0.0, 0.0, R)[0] == pytest.approx(7.5)
    assert reeds_shepp(-7.5, 0.0, 0.0, R)[0] == pytest.approx(7.5)               # straight back
    assert dubins(7.5, 0.0, 0.0, R)[0] == pytest.approx(7.5)
    assert dubins(-0.003, 0.0, 0.0, R)[0] == pytest.approx(2 * np.pi * R + 0.003, abs=1e-4)   # a Dubins car must go around
    assert reeds_shepp(0.0, 0.0, np.pi, R)[0] == pytest.approx(np.pi * R)         # turning on the spot: three arcs of pi/3
    assert dubins(0.0, 2 * R, np.pi, R)[0] == pytest.approx(np.pi * R)            # half circle
    assert reeds_shepp(R, R, np.pi / 2, R)[:2] == (pytest.approx(np.pi * R / 2), 1)   # quarter circle, one maneuver
    # lateral shift: the paper's correcting path of four equal arcs, is a valid path
    y = np.array([0.1, 0.5, 1.0, 2.0, 5.0])
    assert (reeds_shepp(0.0, y, 0.0, R)[0] <= 4 * R * np.arccos(1 - y / (4 * R)) + 1e-9).all()
    rng = np.random.default_rng(3)
    x, y, phi = rng.uniform(-20, 20, 4000), rng.uniform(-20, 20, 4000), rng.uniform(-np.pi, np.pi, 4000)
    L, ns, Lc = reeds_shepp(x, y, phi, R, d_T=2.0)
    D, nd = dubins(x, y, phi, R)
    assert np.isfinite(L).all() and np.isfinite(D).all()
    assert (ns <= 5).all() and (nd <= 3).all()                                    # Corollary 1 l.715, Theorem 2 l.697
    assert (L >= np.hypot(x, y) - 1e-9).all() and (L >= R * np.abs(phi) - 1e-9).all()
    assert (D >= L - 1e-9).all()                                                  # forward-only is a restriction
    assert (Lc >= L + 2.0 - 1e-9).all() and (Lc <= L + 2.0 * ns + 1e-9).all()
    # time flip, reflection (PAPER.md:92 model symmetries), and the metric's symmetry (drive the path backwards from the goal)
    assert np.allclose(reeds_shepp(-x, y, -phi, R)[0], L)
    assert np.allclose(reeds_shepp(x, -y, -phi, R)[0], L)
    c, s = np.cos(phi), np.sin(phi)
    assert np.allclose(reeds_shepp(-(x * c + y * s), x * s - y * c, -phi, R)[0], L)
    assert np.allclose(dubins(x, -y, -phi, R)[0], D)


def test_closed_forms_satisfy_the_dynamic_programming_principle():
    """Completeness of the word families: a shortest-path length f obeys f(goal) <= s + f(goal seen after any
    primitive of length s) and, where f > s, equality for the first primitive of a shortest path.  A family with a
    missing word returns too large a value somewhere, and the inequality fails where a shortest path leaves that region."""
    rng = np.random.default_rng(4)
    n = 30000
    x, y, phi = rng.uniform(-7, 7, n), rng.uniform(-7, 7, n), rng.uniform(-np.pi, np.pi, n)
    L = reeds_shepp(x, y, phi)[0]
    D = dubins(x, y, phi)[0]
    for s in (0.04, 0.35):
        best_rs, best_d = np.full(n, np.inf), np.full(n, np.inf)
        for prim in "LSR":
            for gear in (1.0, -1.0):
                L2 = reeds_shepp(*_seen_after(prim, gear * s, x, y, phi))[0]
                assert (L <= s + L2 + 1e-9).all(), (prim, gear, s)
                best_rs = np.minimum(best_rs, s + L2)
            D2 = dubins(*_seen_after(prim, s, x, y, phi))[0]
            assert (D <= s + D2 + 1e-9).all(), (prim, s)
            best_d = np.minimum(best_d, s + D2)
        if s < 0.1:                                                               # (a switch inside the step costs O(s^2))
            assert (best_rs - L)[L > s].max() < 0.05
            assert np.median((best_d - D)[D > s]) < 1e-6


# ---------------------------------------------------------------------------------------------------------------
# the graph against them
# ---------------------------------------------------------------------------------------------------------------
def free_space(log2_n, log2_nt, R, d_T, flags=0):
    o = oracle.Oracle(log2_n, log2_nt, R, (int(d_T * ONE),) * 6, cost_one_log2=ONE_LOG2, flags=flags, threads=0)
    fp = oracle.Footprint(np.ones((1, 1), np.uint8), 0.0, 0.0)
    C, _ = o.render(fp, np.zeros((o.n, o.n), np.uint8))
    return o, C


def relative(o, start, I, J, T, dx=0.0, dy=0.0):
    """Poses (I, J, T) [+ a world-frame offset in cells] in the frame of the start pose; pose of a vertex by eq (16),
    PAPER.md:256: (i + Psi0(Theta), j + Psi1(Theta), 2 pi Theta / N_theta)."""
    psi = o.psi2.astype(np.float64) / 2.0
    nt = o.nt
    x0, y0 = start[0] + psi[start[2]], start[1] + psi[(start[2] + nt // 4) % nt]
    th0 = 2.0 * np.pi * start[2] / nt
    ex, ey = I + psi[T] + dx - x0, J + psi[(T + nt // 4) % nt] + dy - y0
    c, s = np.cos(th0), np.sin(th0)
    return ex * c + ey * s, -ex * s + ey * c, 2.0 * np.pi * ((T - start[2]) % nt) / nt


def eps_q(v_cells, o, R):
    """Fixed-point rounding of the edge lengths: at most half a cost unit per edge (DESIGN R18)."""
    return 0.5 * (v_cells / min(1.0, 2.0 * np.pi * R / o.nt) + 1.0) / ONE


CASES = [   # log2_n, log2_nt, R, d_T (sufficient: d_T >= 1 + R d_theta + 4R acos(1 - 1/(4R))), forward only
    (7, 6, 8, 10.0, False),
    (7, 7, 16, 14.0, False),
    (7, 6, 8, 10.0, True),
]


@pytest.mark.parametrize("log2_n,log2_nt,R,d_T,fwd", CASES)
def test_free_space_fixpoint_against_the_closed_forms(log2_n, log2_nt, R, d_T, fwd):
    o, C = free_space(log2_n, log2_nt, R, d_T, oracle.FLAG_FORWARD_ONLY if fwd else 0)
    n, nt = o.n, o.nt
    assert d_T >= 1 + R * 2 * np.pi / nt + 4 * R * np.arccos(1 - 1 / (4 * R))      # "sufficient transition costs"
    rng = np.random.default_rng(100 * log2_nt + R)
    h = 0.25                                                                      # sampling pitch of the boxes, cells
    offs = np.arange(-4.0, 4.0 + h / 2, h)
    BX, BY = np.meshgrid(offs, offs, indexing="ij")
    # a box point lies within h/2 per axis of a sample; correcting that costs at most this much
    e = h / np.sqrt(2.0)
    slack = e + 4 * R * np.arccos(1 - e / (4 * R))
    medians = []
    for t0 in (0, 5, nt // 8):                                                    # axis, generic, diagonal start headings
        start = (n // 2, n // 2, t0)
        V = o.dijkstra(C, None, start, "star")
        K = 60
        I = rng.integers(n // 2 - 24, n // 2 + 25, K)
        J = rng.integers(n // 2 - 24, n // 2 + 25, K)
        T = rng.integers(0, nt, K)
        assert (V[T, J, I] != INF).all()
        v = V[T, J, I].astype(np.float64) / ONE
        gx, gy, gp = relative(o, start, I, J, T)
        if fwd:
            L, ns = dubins(gx, gy, gp, R)
            Lc = L + d_T * ns
        else:
            L, ns, Lc = reeds_shepp(gx, gy, gp, R, d_T)
        # (1) typical case: the graph value IS the closed form, up to snapping (not a theorem: the outliers are one
        #     transition cost up, where snapping needs a correcting maneuver, or one or two down, where it saves one)
        medians.append(np.median(np.abs(v - Lc)))
        # (2) Theorem 7 (graph not too pessimistic): continuum reach within d = Lc => some vertex within
        #     7 + pi d / N_theta cells and 4 angular cells has V <= d
        for k in range(K):
            d = Lc[k]
            r = int(np.floor(7 + np.pi * d / nt))
            ii = np.arange(max(I[k] - r, 0), min(I[k] + r, n - 1) + 1)
            jj = np.arange(max(J[k] - r, 0), min(J[k] + r, n - 1) + 1)
            tt = np.arange(T[k] - 4, T[k] + 5) % nt
            box = V[np.ix_(tt, jj, ii)].astype(np.float64) / ONE
            assert box.min() <= d + eps_q(d, o, R), (start, I[k], J[k], T[k], box.min(), d)
        # (3) Theorem 6 (graph not too optimistic).  Its proof (Corollary 2 l.787, Lemmas 4-5): a graph path of m
        #     maneuvers has a continuum twin of the same length ending within ceil(3m/2)/2 cells, same angle.  So
        #     V >= min over m of m d_T + (shortest continuum path into that box); m >= 6 is bounded by 6 d_T alone.
        #     The literal statement (4 cells, one transition cost) follows and is asserted too.
        #     (forward only: the twin is a Reeds-Shepp path as well; Dubins lengths are discontinuous and allow no sampling bound)
        sub = rng.choice(K, 24, replace=False)
        for k in sub:
            bx, by, bp = relative(o, start, I[k], J[k], T[k], BX, BY)
            box_L = reeds_shepp(bx, by, np.full_like(bx, bp), R)[0]
            rad = np.maximum(np.abs(BX), np.abs(BY))
            lb = 6 * d_T
            for m in range(1, 6):
                lb = min(lb, m * d_T + box_L[rad <= np.ceil(1.5 * m) / 2 + 1e-9].min() - slack)
            assert v[k] >= lb - eps_q(v[k], o, R), (start, I[k], J[k], T[k], v[k], lb)
            assert v[k] >= box_L.min() + d_T - slack - eps_q(v[k], o, R)
    assert max(medians) <= 1.0, medians                                           # cells; observed 0.3 - 0.6
