"""Pins for the oracle's obstacle rendering.

The rasterisation rule (DESIGN R15) is our own definition -- the paper gives none -- so it is "parity
unpinned" against the paper; what is pinned here is that the oracle implements the configuration-space
obstacle of PAPER.md:88 ("the vehicle shape ... transformed into world coordinates intersects an obstacle"):
exact box dilation at the axis angles, a rotated-rectangle test at every angle up to one pixel of boundary,
monotonicity in the footprint, area preservation, and the wall / seam of PAPER.md:226.
"""
import numpy as np
import pytest

import oracle
import scenes


def make(log2_n=5, log2_nt=5, R=4):
    return oracle.Oracle(log2_n, log2_nt, R, (4096,) * 6)


def test_axis_angles_are_exact_box_dilations():
    o = make()
    n, nt = o.n, o.nt
    L, W = 6, 3
    fp = oracle.Footprint.box(L, W)
    rng = np.random.default_rng(3)
    hard = (rng.random((n, n)) < 0.03).astype(np.uint8)
    soft = rng.integers(16, 200, size=(n, n)).astype(np.uint8)
    C, S = o.render(fp, hard, soft, method="brute")
    H = hard.astype(bool).copy()
    H[0, :] = True
    H[:, 0] = True
    assert (o.psi2[[0, nt // 4, nt // 2, 3 * nt // 4]] == 0).all()        # integer R: no half-cell offset there
    # vehicle rectangle u in [-0.2L, 0.8L) = {-1..4}, v in [-W/2, W/2) = {-1, 0, 1} for L=6, W=3
    us, vs = range(-1, 5), range(-1, 2)
    for t, (ux, uy, vx, vy) in {0: (1, 0, 0, 1), nt // 4: (0, 1, -1, 0), nt // 2: (-1, 0, 0, -1), 3 * nt // 4: (0, -1, 1, 0)}.items():
        want_c = np.zeros((n, n), bool)
        want_s = np.zeros((n, n), np.uint8)
        for u in us:
            for v in vs:
                da, db = u * ux + v * vx, u * uy + v * vy                    # PAPER.md:86 with cos, sin in {0, +-1}
                want_c |= np.roll(H, (-db, -da), axis=(0, 1))
                want_s = np.maximum(want_s, np.roll(soft, (-db, -da), axis=(0, 1)))
        want_c[0, :] = True
        want_c[:, 0] = True
        assert (C[t].astype(bool) == want_c).all(), t
        assert (S[t] == np.maximum(want_s, 16)).all(), t


def test_every_angle_matches_a_rotated_rectangle_up_to_the_boundary():
    """Pixels whose centre is well inside the rotated L x W rectangle (by more than the fixed-point and
    half-pixel slack) are covered; pixels well outside are not; the covered area is L*W within 12 %."""
    o = make(6, 6, 8)
    L, W = 10, 5
    fp = oracle.Footprint.box(L, W)
    psi2, nt = o.psi2, o.nt
    for t in range(nt):
        da, db = o.footprint_offsets(fp, t)
        got = set(zip(da.tolist(), db.tolist()))
        assert abs(len(got) - L * W) <= 0.12 * L * W
        th = 2 * np.pi * t / nt
        x0, y0 = psi2[t] / 2.0, psi2[(t + nt // 4) % nt] / 2.0
        for a in range(-14, 15):
            for b in range(-14, 15):
                u = (a - x0) * np.cos(th) + (b - y0) * np.sin(th)
                v = -(a - x0) * np.sin(th) + (b - y0) * np.cos(th)
                inside = min(u + 0.2 * L, 0.8 * L - u, v + W / 2, W / 2 - v)   # signed distance to the rectangle edge
                if inside > 0.02:
                    assert (a, b) in got
                if inside < -0.02:
                    assert (a, b) not in got


def test_monotone_in_footprint_and_in_obstacles():
    o = make()
    n = o.n
    rng = np.random.default_rng(4)
    hard = (rng.random((n, n)) < 0.02).astype(np.uint8)
    soft = rng.integers(16, 255, size=(n, n)).astype(np.uint8)
    small = oracle.Footprint.box(4, 2)
    big = oracle.Footprint(np.ones((4, 6), np.uint8), small.ou + 1, small.ov + 1)   # small padded by one pixel all round
    Cs, Ss = o.render(small, hard, soft, method="brute")
    Cb, Sb = o.render(big, hard, soft, method="brute")
    assert (Cs <= Cb).all() and (Ss <= Sb).all() and Cb.sum() > Cs.sum()
    more = hard.copy()
    more[10:12, 20:25] = 1
    Cm, _ = o.render(small, more, soft, method="brute")
    assert (Cs <= Cm).all()
    # C = 1 and soft >= the soft value under the rear axle; S >= 16 everywhere
    assert Ss.min() >= 16


@pytest.mark.parametrize("seed,vehicle,soft", [(1, (4, 2), True), (2, (7, 3), True), (3, (5, 5), False)])
def test_run_renderer_equals_brute_force(seed, vehicle, soft):
    sc = scenes.random_scene(5, 6, 6, seed, vehicle=vehicle, soft=soft)
    o = oracle.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct)
    fp = oracle.Footprint(sc.mask, sc.ou, sc.ov)
    Cb, Sb = o.render(fp, sc.hard, sc.soft, method="brute")
    Cr, Sr = o.render(fp, sc.hard, sc.soft, method="runs")
    assert (Cb == Cr).all()
    if soft:
        assert (Sb == Sr).all()
    # a non-convex mask with holes (arbitrary shape, Figure 6)
    m = np.ones((5, 7), np.uint8)
    m[1:4, 2:5] = 0
    m[2, :] = [1, 0, 0, 1, 0, 0, 1]
    fp2 = oracle.Footprint(m, 1.7, 2.0)
    Cb, Sb = o.render(fp2, sc.hard, sc.soft, method="brute")
    Cr, Sr = o.render(fp2, sc.hard, sc.soft, method="runs")
    assert (Cb == Cr).all() and (Sb is None or (Sb == Sr).all())
    # single poses agree with the volume
    rng = np.random.default_rng(seed)
    for _ in range(50):
        i, j, t = (int(rng.integers(o.n)), int(rng.integers(o.n)), int(rng.integers(o.nt)))
        c, s = o.render_pose(fp2, sc.hard, sc.soft, i, j, t)
        assert c == Cb[t, j, i] and (Sb is None or s == Sb[t, j, i])
    # ... and so do single planes (the form the full-size GPU tests use)
    for t in (0, o.nt // 8, o.nt - 3):
        Cp, Sp = o.render_plane(fp2, sc.hard, sc.soft, t)
        assert (Cp == Cb[t]).all() and (Sb is None or (Sp == Sb[t]).all())


def test_run_renderer_equals_brute_force_with_a_large_footprint():
    """The vehicle of config 5 (44 x 20 cells: footprint radius 38, runs up to 44 cells long, i.e. every level of the sparse
    tables of row maxima / prefix counts up to 2^5) on a small grid, whole volume against the plain O(N_R |box|) loop."""
    for vehicle, seed in (((44, 20), 41),):
        sc = scenes.random_scene(7, 4, 2.4, seed, vehicle=vehicle, n_rects=14, max_side=9, soft=True)
        o = oracle.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct)
        fp = oracle.Footprint(sc.mask, sc.ou, sc.ov)
        Cb, Sb = o.render(fp, sc.hard, sc.soft, method="brute")
        Cr, Sr = o.render(fp, sc.hard, sc.soft, method="runs")
        assert (Cb == Cr).all() and (Sb == Sr).all()
        assert 0 < Cb.mean() < 1


def test_footprint_overhanging_the_seam_is_blocked():
    """PAPER.md:226 + DESIGN R13: image addressing is toroidal and the pixels a = 0, b = 0 are hard."""
    o = make()
    n, nt = o.n, o.nt
    fp = oracle.Footprint.box(6, 3)
    C, _ = o.render(fp, np.zeros((n, n), np.uint8), None, method="brute")
    assert C[:, 0, :].all() and C[:, :, 0].all()
    assert C[0, 16, n - 4] == 1 and C[0, 16, n - 6] == 0      # nose at i+4 reaches column 0 (= n) or not
    assert C[nt // 2, 16, 4] == 1 and C[nt // 2, 16, 6] == 0  # heading -x
    assert C[0, 16, 1] == 1 and C[0, 16, 2] == 0              # tail at i-1
