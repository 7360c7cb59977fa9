"""Closed-form shortest paths of the Dubins and Reeds-Shepp vehicles in free space (tests only).

Written from the mathematics, independent of oracle/ and of the CUDA path: a path is a word of segments
(L = left arc, R = right arc, S = straight; signed length, negative = reverse gear) on unit turn radius, start at
(0, 0, heading 0).  PAPER.md:697 (Theorem 2, Dubins: CSC, CCC) and PAPER.md:703-715 (Theorem 3 / Corollary 1,
Reeds-Shepp: at most five segments, at most two cusps) name the sufficient families; the segment lengths of every
word follow from the circle-centre geometry.  Nothing here is trusted because it was typed: `endpoint()` integrates
every candidate word forward and a candidate that does not land on the goal is discarded, so every reported length is
the length of a real path (an upper bound of the optimum); tests/test_closed_forms.py then pins the families as
COMPLETE through the dynamic-programming principle, known values and the metric axioms.

Everything is vectorised over numpy arrays of goals.
"""
import numpy as np

PI = np.pi
TOL = 1e-7


def mod2pi(a):
    """Wrap to (-pi, pi]."""
    return a - 2.0 * PI * np.ceil((a - PI) / (2.0 * PI))


def polar(x, y):
    return np.hypot(x, y), np.arctan2(y, x)


def endpoint(word, lengths):
    """Integrate a word forward from (0, 0, 0).  word: string over 'LRS'; lengths: list of arrays (signed)."""
    x = np.zeros_like(lengths[0], dtype=np.float64)
    y = np.zeros_like(x)
    th = np.zeros_like(x)
    for c, s in zip(word, lengths):
        if c == "S":
            x = x + s * np.cos(th)
            y = y + s * np.sin(th)
        elif c == "L":                      # centre (x - sin th, y + cos th)
            t2 = th + s
            x = x + np.sin(t2) - np.sin(th)
            y = y - np.cos(t2) + np.cos(th)
            th = t2
        else:                               # 'R': centre (x + sin th, y - cos th)
            t2 = th - s
            x = x - np.sin(t2) + np.sin(th)
            y = y + np.cos(t2) - np.cos(th)
            th = t2
    return x, y, th


def _accept(word, lengths, x, y, phi):
    """Total length of the candidate where it really ends at the goal, +inf elsewhere; and its number of maneuvers
    (segments of non-zero length; two consecutive arcs of the same hand and gear would count once, no word has them)."""
    ls = [np.where(np.isfinite(s), s, 0.0) for s in lengths]
    ex, ey, eth = endpoint(word, ls)
    ok = np.ones_like(x, dtype=bool)
    for s in lengths:
        ok &= np.isfinite(s)
    ok &= (np.abs(ex - x) < 1e-6) & (np.abs(ey - y) < 1e-6) & (np.abs(mod2pi(eth - phi)) < 1e-6)
    total = sum(np.abs(s) for s in ls)
    nseg = sum((np.abs(s) > 1e-9).astype(np.int64) for s in ls)
    return np.where(ok, total, np.inf), nseg


# ------------------------------------------------------------------------------------------------------------------
# Dubins (forward only): LSL, RSR, LSR, RSL, LRL, RLR.  PAPER.md:697 (Theorem 2).
# ------------------------------------------------------------------------------------------------------------------
def _wrap_pos(a):
    """Wrap to [0, 2 pi): an arc driven forward."""
    a = np.mod(a, 2.0 * PI)
    return np.where(a >= 2.0 * PI - 1e-12, 0.0, a)


def _dubins_words(x, y, phi):
    """Yield (word, [lengths]) for the L-first words; the R-first ones follow by reflection."""
    # the start circle to the left has its centre at (0, 1), the goal circle to the left at (x - sin phi, y + cos phi),
    # the goal circle to the right at (x + sin phi, y - cos phi)
    # LSL: outer tangent, heading of the straight = direction between the centres
    dx, dy = x - np.sin(phi), y + np.cos(phi) - 1.0
    d, a = polar(dx, dy)
    yield "LSL", [_wrap_pos(a), d, _wrap_pos(phi - a)]
    # LSR: inner tangent; centres D apart, straight sqrt(D^2 - 4), heading = direction of centres + asin(2 / D)
    dx, dy = x + np.sin(phi), y - np.cos(phi) - 1.0
    D, a = polar(dx, dy)
    with np.errstate(invalid="ignore"):
        s = np.sqrt(D * D - 4.0)
        psi = a + np.arctan2(2.0, s)
    yield "LSR", [_wrap_pos(psi), s, _wrap_pos(psi - phi)]
    # LRL: middle circle touches both, its centre 2 away from each; two mirror solutions
    dx, dy = x - np.sin(phi), y + np.cos(phi) - 1.0
    D, a = polar(dx, dy)
    with np.errstate(invalid="ignore"):
        g = np.arccos(D / 4.0)              # angle at the start centre between the centre line and the middle centre
    for sg in (1.0, -1.0):
        # direction start centre -> middle centre is a + sg g; the car is at angle (heading - pi/2) on its left circle
        t = _wrap_pos(a + sg * g + PI / 2.0)
        u = _wrap_pos(sg * (PI - 2.0 * g) if sg > 0 else PI + 2.0 * g)
        # on leaving the middle (right) circle the heading is t - u; the last arc brings it to phi
        v = _wrap_pos(phi - (t - u))
        yield "LRL", [t, u, v]
        yield "LRL", [t, _wrap_pos(2.0 * PI - u), _wrap_pos(phi - (t - (2.0 * PI - u)))]


def dubins(x, y, phi, R=1.0):
    """(length, n_maneuvers) of the shortest Dubins path from (0, 0, 0) to (x, y, phi); arrays, turn radius R."""
    x, y, phi = np.broadcast_arrays(np.asarray(x, float) / R, np.asarray(y, float) / R, np.asarray(phi, float))
    best = np.full(x.shape, np.inf)
    nseg = np.zeros(x.shape, np.int64)
    for refl in (False, True):
        yy, pp = (-y, -phi) if refl else (y, phi)
        for word, ls in _dubins_words(x, yy, pp):
            w = word.translate(str.maketrans("LR", "RL")) if refl else word
            tot, ns = _accept(w, ls, x, y, phi)
            better = tot < best - 1e-12
            best = np.where(better, tot, best)
            nseg = np.where(better, ns, nseg)
    return best * R, nseg


# ------------------------------------------------------------------------------------------------------------------
# Reeds-Shepp.  PAPER.md:703-715 (Theorem 3, Corollary 1): C|C_{pi/2}SC_{pi/2}|C, CSC, C|C|C, CC|C, C|CC, CCu|CuC,
# C|CuCu|C and their sub-words.  Base words start with a forward left arc; the others follow from the symmetries
#   time flip  (x, y, phi) -> (-x, y, -phi)                     every gear reversed
#   reflection (x, y, phi) -> (x, -y, -phi)                     L <-> R
#   backwards  (x, y, phi) -> (x cos phi + y sin phi, x sin phi - y cos phi, phi)    word read from its end
# ------------------------------------------------------------------------------------------------------------------
def _nan_where(cond, a):
    return np.where(cond, a, np.nan)


def _tau_omega(u, v, xi, eta, phi):
    delta = mod2pi(u - v)
    A = np.sin(u) - np.sin(delta)
    B = np.cos(u) - np.cos(delta) - 1.0
    t1 = np.arctan2(eta * A - xi * B, xi * A + eta * B)
    t2 = 2.0 * (np.cos(delta) - np.cos(v) - np.cos(u)) + 3.0
    tau = np.where(t2 < 0, mod2pi(t1 + PI), mod2pi(t1))
    omega = mod2pi(tau - u + v - phi)
    return tau, omega


def _rs_base_words(x, y, phi):
    """Yield (word, [signed lengths]) of the base words for goal (x, y, phi); invalid entries are NaN."""
    with np.errstate(invalid="ignore", divide="ignore"):
        # L+ S+ L+
        u, t = polar(x - np.sin(phi), y - 1.0 + np.cos(phi))
        v = mod2pi(phi - t)
        ok = (t >= -TOL) & (v >= -TOL)
        yield "LSL", [_nan_where(ok, t), u, v]
        # L+ S+ R+
        u1, t1 = polar(x + np.sin(phi), y - 1.0 - np.cos(phi))
        u = np.sqrt(u1 * u1 - 4.0)
        th = np.arctan2(2.0, u)
        t = mod2pi(t1 + th)
        v = mod2pi(t - phi)
        ok = (t >= -TOL) & (v >= -TOL)
        yield "LSR", [_nan_where(ok, t), u, v]
        # L+ R- L(+-)
        xi, eta = x - np.sin(phi), y - 1.0 + np.cos(phi)
        u1, th = polar(xi, eta)
        u = -2.0 * np.arcsin(0.25 * u1)
        t = mod2pi(th + 0.5 * u + PI)
        v = mod2pi(phi - t + u)
        ok = (u1 <= 4.0) & (t >= -TOL) & (u <= TOL)
        yield "LRL", [_nan_where(ok, t), u, v]
        # L+ R+u L-u R-
        xi, eta = x + np.sin(phi), y - 1.0 - np.cos(phi)
        rho = 0.25 * (2.0 + np.hypot(xi, eta))
        u = np.arccos(rho)
        t, v = _tau_omega(u, -u, xi, eta, phi)
        ok = (rho <= 1.0) & (t >= -TOL) & (v <= TOL)
        yield "LRLR", [_nan_where(ok, t), u, -u, v]
        # L+ R-u L-u R+
        rho = (20.0 - xi * xi - eta * eta) / 16.0
        u = -np.arccos(rho)
        t, v = _tau_omega(u, u, xi, eta, phi)
        ok = (rho >= 0.0) & (rho <= 1.0) & (u >= -0.5 * PI - TOL) & (t >= -TOL) & (v >= -TOL)
        yield "LRLR", [_nan_where(ok, t), u, u, v]
        # L+ R-(pi/2) S- L-
        xi, eta = x - np.sin(phi), y - 1.0 + np.cos(phi)
        rho, th = polar(xi, eta)
        r = np.sqrt(rho * rho - 4.0)
        u = 2.0 - r
        t = mod2pi(th + np.arctan2(r, -2.0))
        v = mod2pi(phi - 0.5 * PI - t)
        ok = (rho >= 2.0) & (t >= -TOL) & (u <= TOL) & (v <= TOL)
        yield "LRSL", [_nan_where(ok, t), np.full_like(t, -0.5 * PI), u, v]
        # L+ R-(pi/2) S- R-
        xi, eta = x + np.sin(phi), y - 1.0 - np.cos(phi)
        rho, th = polar(-eta, xi)
        t = th
        u = 2.0 - rho
        v = mod2pi(t + 0.5 * PI - phi)
        ok = (rho >= 2.0) & (t >= -TOL) & (u <= TOL) & (v <= TOL)
        yield "LRSR", [_nan_where(ok, t), np.full_like(t, -0.5 * PI), u, v]
        # L+ R-(pi/2) S- L-(pi/2) R+
        rho, th = polar(xi, eta)
        u = 4.0 - np.sqrt(rho * rho - 4.0)
        t = mod2pi(np.arctan2((4.0 - u) * xi - 2.0 * eta, -2.0 * xi + (u - 4.0) * eta))
        v = mod2pi(t - phi)
        ok = (rho >= 2.0) & (u <= TOL) & (t >= -TOL) & (v >= -TOL)
        yield "LRSLR", [_nan_where(ok, t), np.full_like(t, -0.5 * PI), u, np.full_like(t, -0.5 * PI), v]


def reeds_shepp(x, y, phi, R=1.0, d_T=0.0):
    """Shortest Reeds-Shepp path from (0, 0, 0) to (x, y, phi) on turn radius R.

    Returns (length, n_maneuvers, with_costs): `length` = min over the words of the path length, `n_maneuvers` the
    maneuver count of that word, `with_costs` = min over the words of length + d_T * n_maneuvers (the best path of
    the Reeds-Shepp family under maneuver-counting transition costs; an UPPER bound of the optimum
    with transition costs, which by Theorem 5 l.751 may also be a non-family path of at most four maneuvers)."""
    x, y, phi = np.broadcast_arrays(np.asarray(x, float) / R, np.asarray(y, float) / R, np.asarray(phi, float))
    x, y, phi = x.copy(), y.copy(), mod2pi(phi)
    best = np.full(x.shape, np.inf)
    nseg = np.zeros(x.shape, np.int64)
    bestc = np.full(x.shape, np.inf)
    dt = d_T / R
    swap = str.maketrans("LR", "RL")
    for back in (False, True):
        if back:
            xb, yb = x * np.cos(phi) + y * np.sin(phi), x * np.sin(phi) - y * np.cos(phi)
        else:
            xb, yb = x, y
        for flip in (False, True):
            for refl in (False, True):
                xx = -xb if flip else xb
                yy = -yb if refl else yb
                pp = -phi if (flip != refl) else phi
                for word, ls in _rs_base_words(xx, yy, pp):
                    w = word.translate(swap) if refl else word
                    ls2 = [-s for s in ls] if flip else list(ls)
                    if back:
                        w, ls2 = w[::-1], ls2[::-1]
                    tot, ns = _accept(w, ls2, x, y, phi)
                    better = tot < best - 1e-12
                    best = np.where(better, tot, best)
                    nseg = np.where(better, ns, nseg)
                    bestc = np.minimum(bestc, tot + dt * ns)
    return best * R, nseg, bestc * R
