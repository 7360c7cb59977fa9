"""Independent Python re-statements used only as pins for the oracle (tests only)."""
import numpy as np

INF = 0xFFFFFFFF
LIMIT = 1 << 30
SF, SB = 1, 4


def sat(x):
    return INF if x >= LIMIT else x


def curve_cells(o, m, c0, c1):
    """Cells of one curve in SWEEP order, as (t, j, i) index tuples."""
    turn = m not in (SF, SB)
    L = o.nt if turn else o.n
    if turn:
        up = m in (0, 2)                                   # LF, RB sweep Theta upward (eq 25, 28)
    else:
        up = (m == SF) == (o.J[c1] > 0)
    ks = range(L) if up else range(L - 1, -1, -1)
    out = []
    for k in ks:
        i, j, t = o.curve_cell(m, c0, c1, k)
        out.append((t, j, i))
    return out


def closed_form_sweep(o, m, V, C, S=None):
    """SURVEY O3 closed form: V'[p] = min(V[p], min over sources s strictly before p on the curve
    (cyclically, less than one lap, for turns) with no blocked cell in [s,p] of
    V[s] + ct + sum_{q in [s,p)} w(q)), all sums saturating at LIMIT."""
    turn = m not in (SF, SB)
    lenq = o.len_q
    ct = o.ct[m]
    Vn = V.copy()
    for c1 in range(o.n if turn else o.nt):
        for c0 in range(o.n):
            cells = curve_cells(o, m, c0, c1)
            L = len(cells)
            for a, p in enumerate(cells):
                if C[p]:
                    continue
                best = int(V[p])
                dist = 0
                for back in range(1, L if turn else a + 1):
                    s = cells[(a - back) % L]
                    if C[s]:
                        break
                    sv = 16 if S is None else int(S[s])
                    dist += (int(lenq[m, s[0]]) * sv) >> 4
                    vs = int(V[s])
                    if vs != INF:
                        best = min(best, sat(vs + ct + dist))
                Vn[p] = best
    return Vn


def random_volume(rng, shape, p_blocked=0.2, p_inf=0.3, vmax=200000):
    C = (rng.random(shape) < p_blocked).astype(np.uint8)
    V = rng.integers(0, vmax, size=shape).astype(np.uint32)
    V[rng.random(shape) < p_inf] = INF
    V[C != 0] = INF
    S = rng.integers(16, 256, size=shape).astype(np.uint8)
    return V, C, S


def pm26_reach(C, start):
    """26-neighbour Piano-mover flood fill on the free cells of C (toroidal), returns step counts."""
    free = C == 0
    dist = np.full(C.shape, -1, np.int64)
    t, j, i = start[2], start[1], start[0]
    front = np.zeros(C.shape, bool)
    front[t, j, i] = True
    dist[t, j, i] = 0
    seen = front.copy()
    d = 0
    while front.any():
        d += 1
        grow = np.zeros_like(front)
        for a in (-1, 0, 1):
            for b in (-1, 0, 1):
                for c in (-1, 0, 1):
                    if a or b or c:
                        grow |= np.roll(front, (a, b, c), axis=(0, 1, 2))
        front = grow & free & ~seen
        dist[front] = d
        seen |= front
    return dist
