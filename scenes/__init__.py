"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests / bench.

This module holds NONE of the method's arithmetic (no tables, no rendering, no sweeps): it only
draws obstacle images, soft-cost images, vehicle masks and start / goal poses with numpy, so that
both sides can be fed identical inputs.  It imports neither `oracle` nor the CUDA package.

The five named configurations are the ones listed in BASELINE.json `configs`; they stand in for
the paper's scene classes (free space, parallel / perpendicular parking, cluttered, maze --
PAPER.md:31, Table 3 l.483-494), whose actual geometry exists only as pictures.  The recipe of
every scene is stated in DESIGN.md section 4.

The soft image follows the paper's pipeline steps 1-2 (distance transform of the
binary obstacle image on the CPU, then "some function of the distance", l.342):
    soft = clip(rint(16 * (1 + 4 / (d + 1))), 16, 255)     (Q4.4 speed-reciprocal, 16 = 1.0)
with d the exact Euclidean distance to the nearest hard pixel.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

LF, SF, RB, RF, SB, LB = range(6)     # maneuver ids in the paper's cycle order


@dataclass
class Scene:
    name: str
    log2_n: int
    log2_nt: int
    R: float
    n_cycles: int
    ct: tuple                      # transition-in cost per maneuver, cost units
    dir_mult: tuple                # Q8.8 per maneuver
    hard: np.ndarray               # uint8 [N][N], row = y (j), col = x (i); non-zero = obstacle
    soft: np.ndarray | None        # uint8 [N][N] Q4.4 or None
    mask: np.ndarray               # uint8 [W][L] vehicle footprint, column p along the length axis
    ou: float                      # fractional origin of the mask (rear-axle centre) in mask pixels
    ov: float
    start: tuple                   # (i, j, Theta)
    goal: tuple
    cost_one_log2: int = 10
    flags: int = 0
    extra_goals: list = field(default_factory=list)

    @property
    def n(self):
        return 1 << self.log2_n

    @property
    def nt(self):
        return 1 << self.log2_nt


def box_mask(length: int, width: int):
    """All-ones L x W mask whose origin puts the rear axle ~21 % from the rear."""
    return np.ones((width, length), np.uint8), 0.2 * length - 0.5, (width - 1) / 2.0


def counting_weights(d_t_cells: float, cost_one_log2: int = 10):
    """Maneuver-counting transition costs: the same d_T on every maneuver."""
    return (int(round(d_t_cells * (1 << cost_one_log2))),) * 6


def soft_from_hard(hard: np.ndarray, k: float = 4.0) -> np.ndarray:
    from scipy import ndimage
    h = hard.astype(bool).copy()
    h[0, :] = True
    h[:, 0] = True
    d = ndimage.distance_transform_edt(~h)
    return np.clip(np.rint(16.0 * (1.0 + k / (d + 1.0))), 16, 255).astype(np.uint8)


def _clearance(hard: np.ndarray) -> np.ndarray:
    """Distance of every pixel to the nearest hard pixel or border wall (toroidal border)."""
    from scipy import ndimage
    n = hard.shape[0]
    h = np.zeros((n + 1, n + 1), bool)
    h[:n, :n] = hard.astype(bool)
    h[0, :] = h[:, 0] = h[n, :] = h[:, n] = True
    return ndimage.distance_transform_edt(~h)[:n, :n]


def _free_pose(rng, clear, r_clear, nt, avoid=None, min_dist=0.0):
    js, is_ = np.nonzero(clear > r_clear)
    assert len(is_) > 0, "no pixel with enough clearance"
    for _ in range(10000):
        k = int(rng.integers(len(is_)))
        i, j = int(is_[k]), int(js[k])
        if avoid is not None and np.hypot(i - avoid[0], j - avoid[1]) < min_dist:
            continue
        return (i, j, int(rng.integers(nt)))
    raise AssertionError("could not place pose")


def _circ_radius(length, width):
    return float(np.hypot(0.8 * length, 0.5 * width) + 2.5)


def _fill_rect(img, x0, y0, w, h):
    n = img.shape[0]
    img[max(0, y0):min(n, y0 + h), max(0, x0):min(n, x0 + w)] = 1


# ---------------------------------------------------------------------------------------------
def config1(seed: int = 1) -> Scene:
    """64^3: free space + 10 random axis-aligned rectangles (3-12 cells per side), vehicle 4x2, R=8, N_T=4."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = 64
    hard = np.zeros((n, n), np.uint8)
    for _ in range(10):
        w, h = int(rng.integers(3, 13)), int(rng.integers(3, 13))
        x0, y0 = int(rng.integers(2, 62 - w + 1)), int(rng.integers(2, 62 - h + 1))
        _fill_rect(hard, x0, y0, w, h)
    mask, ou, ov = box_mask(4, 2)
    clear = _clearance(hard)
    rc = _circ_radius(4, 2)
    start = _free_pose(rng, clear, rc, 64)
    goal = _free_pose(rng, clear, rc, 64, avoid=start, min_dist=8.0)
    return Scene("cfg1_rects_64", 6, 6, 8.0, 4, counting_weights(8), (256,) * 6, hard, None, mask, ou, ov, start, goal)


def config2(seed: int = 2) -> Scene:
    """256^3 parallel parking: curb, two parked 16x7 cars, gap 24 px (1.5 car lengths), R=30, N_T=6."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = 256
    hard = np.zeros((n, n), np.uint8)
    hard[:96, :] = 1                                   # curb band
    _fill_rect(hard, 128 - 12 - 16, 96, 16, 7)         # parked car left of the gap
    _fill_rect(hard, 128 + 12, 96, 16, 7)              # parked car right of the gap
    mask, ou, ov = box_mask(16, 7)
    jit = rng.integers(-2, 3, size=3)
    start = (int(128 - 12 - 40 + jit[0]), int(103 + 14 + jit[1]), int(jit[2]) % 256)
    goal = (123, 99, 0)                                # vehicle centred in the gap, parallel to the curb
    return Scene("cfg2_parallel_256", 8, 8, 30.0, 6, counting_weights(30), (256,) * 6, hard, None, mask, ou, ov, start, goal)


def maze_image(rng, cells=16, pitch=32, wall=4):
    """Recursive-backtracker perfect maze; walls on the low side of every lattice cell."""
    n = cells * pitch
    hard = np.ones((n, n), np.uint8)
    for cy in range(cells):
        for cx in range(cells):
            hard[cy * pitch + wall:(cy + 1) * pitch, cx * pitch + wall:(cx + 1) * pitch] = 0
    seen = np.zeros((cells, cells), bool)
    stack = [(0, 0)]
    seen[0, 0] = True
    while stack:
        cx, cy = stack[-1]
        nb = [(cx + dx, cy + dy) for dx, dy in ((1, 0), (-1, 0), (0, 1), (0, -1))
              if 0 <= cx + dx < cells and 0 <= cy + dy < cells and not seen[cy + dy, cx + dx]]
        if not nb:
            stack.pop()
            continue
        nx, ny = nb[int(rng.integers(len(nb)))]
        if nx != cx:                                   # open the wall strip between the two cells
            x = max(cx, nx) * pitch
            hard[cy * pitch + wall:(cy + 1) * pitch, x:x + wall] = 0
        else:
            y = max(cy, ny) * pitch
            hard[y:y + wall, cx * pitch + wall:(cx + 1) * pitch] = 0
        seen[ny, nx] = True
        stack.append((nx, ny))
    return hard


def config3(seed: int = 3) -> Scene:
    """512^3 maze: 16x16 lattice, walls 4 px, corridors 28 px, vehicle 10x5, R=12, N_T=20."""
    rng = np.random.Generator(np.random.PCG64(seed))
    hard = maze_image(rng)
    mask, ou, ov = box_mask(10, 5)
    c = 4 + 14
    start = (c, c, int(rng.integers(512)))
    goal = (15 * 32 + c, 15 * 32 + c, int(rng.integers(512)))
    extra = [(cx * 32 + c, cy * 32 + c, int(rng.integers(512))) for cx in range(16) for cy in range(16)]
    return Scene("cfg3_maze_512", 9, 9, 12.0, 20, counting_weights(12), (256,) * 6, hard, None, mask, ou, ov,
                 start, goal, extra_goals=extra)


def config4(seed: int = 4) -> Scene:
    """512^3 cluttered lot: 200 oriented rectangles / discs, soft costs, reverse x2, vehicle 20x9, R=40, N_T=8."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = 512
    sx, sy = rng.uniform(60, n - 60, size=2)
    while True:
        gx, gy = rng.uniform(60, n - 60, size=2)
        if np.hypot(gx - sx, gy - sy) >= 300:
            break
    yy, xx = np.mgrid[0:n, 0:n].astype(np.float64)
    hard = np.zeros((n, n), bool)
    for _ in range(200):
        cx, cy = rng.uniform(0, n, size=2)
        if rng.random() < 0.5:
            a, b = rng.uniform(5, 40, size=2)
            th = rng.uniform(0, np.pi)
            u = (xx - cx) * np.cos(th) + (yy - cy) * np.sin(th)
            v = -(xx - cx) * np.sin(th) + (yy - cy) * np.cos(th)
            shape = (np.abs(u) <= a / 2) & (np.abs(v) <= b / 2)
        else:
            r = rng.uniform(3, 15)
            shape = (xx - cx) ** 2 + (yy - cy) ** 2 <= r * r
        hard |= shape
    keep = ((xx - sx) ** 2 + (yy - sy) ** 2 <= 60 ** 2) | ((xx - gx) ** 2 + (yy - gy) ** 2 <= 60 ** 2)
    hard &= ~keep
    hard = hard.astype(np.uint8)
    mask, ou, ov = box_mask(20, 9)
    start = (int(round(sx)), int(round(sy)), int(rng.integers(512)))
    goal = (int(round(gx)), int(round(gy)), int(rng.integers(512)))
    dm = [256] * 6
    dm[LB] = dm[SB] = dm[RB] = 512
    return Scene("cfg4_clutter_512", 9, 9, 40.0, 8, counting_weights(40), tuple(dm), hard, soft_from_hard(hard),
                 mask, ou, ov, start, goal)


def config5(seed: int = 5) -> Scene:
    """1024x1024x512 perpendicular parking lot: 4 rows x 24 stalls (24x48), 70 % occupied, soft costs, R=50, N_T=10."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n, nt = 1024, 512
    hard = np.zeros((n, n), np.uint8)
    x0, y0 = (n - 24 * 24) // 2, (n - (3 * 60 + 4 * 48)) // 2
    row_y = [y0 + 60, y0 + 60 + 48, y0 + 60 + 96 + 60, y0 + 60 + 96 + 60 + 48]
    empty = []
    for r, ry in enumerate(row_y):
        for k in range(24):
            if rng.random() < 0.7:
                _fill_rect(hard, x0 + 24 * k + 2, ry + 2, 20, 44)
            else:
                empty.append((r, k))
    if not empty:
        empty.append((0, 11))
        hard[row_y[0]:row_y[0] + 48, x0 + 24 * 11:x0 + 24 * 12] = 0
    r, k = empty[int(rng.integers(len(empty)))]
    xc = x0 + 24 * k + 12
    if r in (0, 2):                                    # entrance on the low-y side: drive in heading +y
        goal = (xc, row_y[r] + 24 - 13, nt // 4)
    else:                                              # entrance on the high-y side: heading -y
        goal = (xc - 1, row_y[r] + 24 + 13 - 1, 3 * nt // 4)
    start = (x0 + 30, y0 + 30, 0)
    mask, ou, ov = box_mask(44, 20)
    return Scene("cfg5_perp_lot_1024", 10, 9, 50.0, 10, counting_weights(50), (256,) * 6, hard, soft_from_hard(hard),
                 mask, ou, ov, start, goal)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def get_config(k: int) -> Scene:
    return CONFIGS[k](k)


# ---------------------------------------------------------------------------------------------
def random_scene(log2_n, log2_nt, R, seed, n_rects=6, max_side=None, vehicle=(4, 2), soft=False,
                 n_cycles=3, reverse_mult=256, ct=None, flags=0) -> Scene:
    """Small seeded scene for parity tests at arbitrary (also non-cubic) sizes."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n, nt = 1 << log2_n, 1 << log2_nt
    max_side = max_side or max(3, n // 5)
    hard = np.zeros((n, n), np.uint8)
    for _ in range(n_rects):
        w, h = int(rng.integers(1, max_side + 1)), int(rng.integers(1, max_side + 1))
        _fill_rect(hard, int(rng.integers(1, n - w)), int(rng.integers(1, n - h)), w, h)
    mask, ou, ov = box_mask(*vehicle)
    clear = _clearance(hard)
    rc = _circ_radius(*vehicle)
    if not (clear > rc).any():
        hard[:] = 0
        clear = _clearance(hard)
    start = _free_pose(rng, clear, rc, nt)
    goal = _free_pose(rng, clear, rc, nt)
    dm = [256] * 6
    dm[LB] = dm[SB] = dm[RB] = reverse_mult
    return Scene(f"rand_{log2_n}_{log2_nt}_{seed}", log2_n, log2_nt, float(R), n_cycles,
                 tuple(ct) if ct is not None else counting_weights(R), tuple(dm), hard,
                 soft_from_hard(hard) if soft else None, mask, ou, ov, start, goal, flags=flags)


def random_lane_map(n: int, seed: int, max_pen: int = 80):
    """Lane map for parity tests (DESIGN R28): piecewise-constant 8 x 8 blocks of random preferred headings and Q4.4 factors
    (a quarter of the blocks carry no penalty, a few carry factors below 16, which count as 16)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    b = max(1, n // 8)
    d = np.kron(rng.integers(0, 256, size=(8, 8)), np.ones((b, b), np.int64)).astype(np.uint8)
    pen = rng.integers(8, max_pen + 1, size=(8, 8))
    pen[rng.random((8, 8)) < 0.25] = 16
    return np.ascontiguousarray(d[:n, :n]), np.ascontiguousarray(np.kron(pen, np.ones((b, b), np.int64)).astype(np.uint8)[:n, :n])


def two_lane_road(log2_n: int = 9, log2_nt: int = 9, seed: int = 6):
    """A scene shaped like Figure 19 ('penalties to inform the planner not to use the reverse direction lane
    and stay to the right'): a horizontal two-lane road across the grid between two walls with a few parked boxes along its
    edges; the lower lane (smaller y) runs towards +x, the upper lane towards -x, driving a lane the wrong way costs a factor 4,
    and a strip along the centre line costs 1.5 whichever way one faces (an area penalty: lane_pen 24 with the heading of the
    lane it lies in).  Vehicle 20 x 9, R = 40 at 512 (scaled with N), N_T = 6, reverse x2; start in the lower lane at the left
    facing +x, goal in the upper lane at the left facing -x (a U-turn further down the road), extra goals along both lanes.
    -> (Scene, lane_dir, lane_pen)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n, nt = 1 << log2_n, 1 << log2_nt
    s = n / 512.0
    L, W, R = max(4, int(round(20 * s))), max(2, int(round(9 * s))), max(4.0, 40.0 * s)
    half = int(round(70 * s))                                   # half width of the road
    mid = n // 2
    hard = np.zeros((n, n), np.uint8)
    hard[: mid - half, :] = 1
    hard[mid + half:, :] = 1
    for _ in range(6):                                          # parked boxes along the kerbs
        x0 = int(rng.integers(int(40 * s), n - int(60 * s)))
        if rng.random() < 0.5:
            _fill_rect(hard, x0, mid - half, L + 2, W + 1)
        else:
            _fill_rect(hard, x0, mid + half - W - 1, L + 2, W + 1)
    lane_dir = np.zeros((n, n), np.uint8)
    lane_dir[mid:, :] = 128                                     # upper lane: heading -x
    lane_pen = np.full((n, n), 64, np.uint8)                    # x4 against the lane
    strip = max(1, int(round(4 * s)))
    lane_pen[mid - strip: mid + strip, :] = 24
    lane_dir[mid - strip: mid, :] = 128                         # the centre strip is charged to whoever drives ALONG it: its
    lane_dir[mid: mid + strip, :] = 0                           # 'preferred' heading is the opposite lane's
    mask, ou, ov = box_mask(L, W)
    soft = soft_from_hard(hard)
    y_lo, y_hi = mid - half // 2, mid + half // 2
    start = (int(60 * s), y_lo, 0)
    goal = (int(60 * s), y_hi, nt // 2)
    extra = [(int(x), y_lo, 0) for x in np.linspace(100 * s, n - 60 * s, 6)] + [(int(x), y_hi, nt // 2) for x in np.linspace(100 * s, n - 60 * s, 6)]
    dm = [256] * 6
    dm[LB] = dm[SB] = dm[RB] = 512
    sc = Scene(f"two_lane_road_{n}", log2_n, log2_nt, float(R), 6, counting_weights(R / 4), tuple(dm), hard, soft, mask, ou, ov,
               start, goal, extra_goals=extra)
    return sc, lane_dir, lane_pen
