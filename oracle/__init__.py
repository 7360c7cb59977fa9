"""TEST INFRASTRUCTURE ONLY -- ctypes front-end of the plain CPU oracle (oracle/nhp_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2306_01301_b200 (the CUDA path) and the CUDA path
never imports it.  All arithmetic of the method lives in nhp_oracle.c; this file only marshals
numpy arrays.  Citations are PAPER.md line numbers (see nhp_oracle.c for the full header).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nhp_oracle.c")
_LIB = os.path.join(_HERE, "libnhp_oracle.so")

INF = 0xFFFFFFFF
LIMIT = 1 << 30
FLAG_FORWARD_ONLY = 1
LF, SF, RB, RF, SB, LB = range(6)          # cycle order
MANEUVER_NAMES = ("LF", "SF", "RB", "RF", "SB", "LB")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no CUDA involved)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Params(C.Structure):
    _fields_ = [("log2_n", C.c_int32), ("log2_nt", C.c_int32), ("R", C.c_double),
                ("ct", C.c_uint32 * 6), ("dir_mult", C.c_uint32 * 6),
                ("cost_one_log2", C.c_int32), ("flags", C.c_int32)]


class _Footprint(C.Structure):
    _fields_ = [("mask", C.c_void_p), ("mw", C.c_int32), ("mh", C.c_int32),
                ("ou", C.c_double), ("ov", C.c_double)]


class _Waypoint(C.Structure):
    _fields_ = [("i", C.c_int32), ("j", C.c_int32), ("theta", C.c_int32), ("m", C.c_int32)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Params), C.POINTER(C.c_int)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_get_threads.argtypes = [C.c_void_p]
        for name in ("beta", "psi2", "I", "J", "K", "B", "len_q", "cosq", "sinq"):
            f = getattr(L, "orc_" + name)
            f.restype = C.c_void_p
            f.argtypes = [C.c_void_p]
        L.orc_curve_cell.argtypes = [C.c_void_p] + [C.c_int] * 4 + [C.POINTER(C.c_int)] * 3
        L.orc_edge.argtypes = [C.c_void_p] + [C.c_int] * 4 + [C.POINTER(C.c_int)] * 3
        L.orc_footprint_radius.argtypes = [C.POINTER(_Footprint)]
        L.orc_render_pose.argtypes = [C.c_void_p, C.POINTER(_Footprint), C.c_void_p, C.c_void_p,
                                      C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_render_brute.argtypes = [C.c_void_p, C.POINTER(_Footprint)] + [C.c_void_p] * 4
        L.orc_render_brute_plane.argtypes = [C.c_void_p, C.POINTER(_Footprint), C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_apply_lane.argtypes = [C.c_void_p] * 4
        L.orc_apply_lane.restype = None
        L.orc_render_runs.argtypes = [C.c_void_p, C.POINTER(_Footprint)] + [C.c_void_p] * 4
        L.orc_footprint_offsets.argtypes = [C.c_void_p, C.POINTER(_Footprint), C.c_int, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_sweep.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_cycles.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_run.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p] + [C.c_int] * 4
        L.orc_dijkstra.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p] + [C.c_int] * 3 + [C.c_void_p]
        L.orc_backtrack.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p] + [C.c_int] * 6 + \
            [C.POINTER(_Waypoint), C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_uint32)]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"oracle {what} failed with code {code}")
        self.code = code


class Footprint:
    """Binary vehicle mask with fractional origin (DESIGN R15).  mask[q, p]: p along the length axis."""

    def __init__(self, mask: np.ndarray, ou: float, ov: float):
        self.mask = np.ascontiguousarray(mask, dtype=np.uint8)
        assert self.mask.ndim == 2
        self.ou, self.ov = float(ou), float(ov)
        self._c = _Footprint(self.mask.ctypes.data, self.mask.shape[1], self.mask.shape[0], self.ou, self.ov)

    @staticmethod
    def box(length: int, width: int) -> "Footprint":
        """L x W rectangle u in [-0.2L, 0.8L), v in [-W/2, W/2): rear axle ~21 % from the rear."""
        return Footprint(np.ones((width, length), np.uint8), 0.2 * length - 0.5, (width - 1) / 2.0)

    def radius(self) -> int:
        return _load().orc_footprint_radius(C.byref(self._c))


class Oracle:
    """Tables + sweeps + Dijkstra + back-tracking on one (N, N, N_theta) grid."""

    def __init__(self, log2_n, log2_nt, R, ct, dir_mult=(256,) * 6, cost_one_log2=10, flags=0, threads=1):
        L = _load()
        p = _Params(log2_n, log2_nt, float(R), (C.c_uint32 * 6)(*ct), (C.c_uint32 * 6)(*dir_mult), cost_one_log2, flags)
        err = C.c_int(0)
        self._h = L.orc_create(C.byref(p), C.byref(err))
        if not self._h:
            raise OracleError(err.value, "create")
        self.n, self.nt = 1 << log2_n, 1 << log2_nt
        self.ct, self.dir_mult, self.flags = tuple(ct), tuple(dir_mult), flags
        self.shape = (self.nt, self.n, self.n)
        self.set_threads(threads)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.orc_destroy(self._h)
            self._h = None

    def set_threads(self, t):
        _load().orc_set_threads(self._h, int(t))

    @property
    def threads(self):
        return _load().orc_get_threads(self._h)

    def _table(self, name, dtype, shape):
        addr = getattr(_load(), "orc_" + name)(self._h)
        n = int(np.prod(shape))
        buf = (C.c_char * (n * np.dtype(dtype).itemsize)).from_address(addr)
        return np.frombuffer(buf, dtype=dtype).reshape(shape).copy()

    @property
    def beta(self): return self._table("beta", np.int32, (self.nt,))
    @property
    def psi2(self): return self._table("psi2", np.uint8, (self.nt,))
    @property
    def I(self): return self._table("I", np.uint8, (self.nt,))
    @property
    def J(self): return self._table("J", np.int8, (self.nt,))
    @property
    def K(self): return self._table("K", np.float64, (self.nt,))
    @property
    def B(self): return self._table("B", np.int32, (self.nt, self.n))
    @property
    def len_q(self): return self._table("len_q", np.uint32, (6, self.nt))
    @property
    def cosq(self): return self._table("cosq", np.int32, (self.nt,))
    @property
    def sinq(self): return self._table("sinq", np.int32, (self.nt,))

    def curve_cell(self, m, c0, c1, k):
        i, j, t = C.c_int(), C.c_int(), C.c_int()
        _load().orc_curve_cell(self._h, m, c0, c1, k, C.byref(i), C.byref(j), C.byref(t))
        return i.value, j.value, t.value

    def edge(self, m, i, j, t):
        a, b, c = C.c_int(), C.c_int(), C.c_int()
        _load().orc_edge(self._h, m, i, j, t, C.byref(a), C.byref(b), C.byref(c))
        return a.value, b.value, c.value

    # ---- rendering -------------------------------------------------------------------
    def _imgs(self, hard, soft):
        hard = np.ascontiguousarray(hard, np.uint8)
        assert hard.shape == (self.n, self.n)
        if soft is not None:
            soft = np.ascontiguousarray(soft, np.uint8)
            assert soft.shape == (self.n, self.n)
        return hard, soft

    def render_pose(self, fp: Footprint, hard, soft, i, j, t):
        hard, soft = self._imgs(hard, soft)
        c, s = C.c_uint8(), C.c_uint8()
        rc = _load().orc_render_pose(self._h, C.byref(fp._c), _ptr(hard), _ptr(soft), i, j, t, C.byref(c), C.byref(s))
        if rc:
            raise OracleError(rc, "render_pose")
        return c.value, s.value

    def render(self, fp: Footprint, hard, soft=None, method="runs"):
        """-> (C uint8 {0,1} [Theta][j][i], S uint8 Q4.4 or None)."""
        hard, soft = self._imgs(hard, soft)
        Cv = np.empty(self.shape, np.uint8)
        Sv = np.empty(self.shape, np.uint8) if soft is not None else None
        f = _load().orc_render_brute if method == "brute" else _load().orc_render_runs
        rc = f(self._h, C.byref(fp._c), _ptr(hard), _ptr(soft), _ptr(Cv), _ptr(Sv))
        if rc:
            raise OracleError(rc, "render")
        return Cv, Sv

    def render_plane(self, fp: Footprint, hard, soft, t):
        """Plane t of the brute-force rendering -> (C uint8 [j][i], S uint8 or None)."""
        hard, soft = self._imgs(hard, soft)
        Cp = np.empty((self.n, self.n), np.uint8)
        Sp = np.empty((self.n, self.n), np.uint8) if soft is not None else None
        rc = _load().orc_render_brute_plane(self._h, C.byref(fp._c), _ptr(hard), _ptr(soft), int(t), _ptr(Cp), _ptr(Sp))
        if rc:
            raise OracleError(rc, "render_plane")
        return Cp, Sp

    def apply_lane(self, Sv, lane_dir, lane_pen):
        """Area / orientation penalty of DESIGN R28 folded into the soft volume Sv (uint8 [Theta][j][i]) in place; returns Sv."""
        assert Sv.dtype == np.uint8 and Sv.flags.c_contiguous and Sv.shape == self.shape
        lane_dir, lane_pen = np.ascontiguousarray(lane_dir, np.uint8), np.ascontiguousarray(lane_pen, np.uint8)
        assert lane_dir.shape == (self.n, self.n) and lane_pen.shape == (self.n, self.n)
        _load().orc_apply_lane(self._h, _ptr(Sv), _ptr(lane_dir), _ptr(lane_pen))
        return Sv

    def footprint_offsets(self, fp: Footprint, t):
        cap = (2 * fp.radius() + 1) ** 2
        da, db = np.empty(cap, np.int32), np.empty(cap, np.int32)
        cnt = _load().orc_footprint_offsets(self._h, C.byref(fp._c), t, _ptr(da), _ptr(db), cap)
        return da[:cnt].copy(), db[:cnt].copy()

    # ---- graph processing -------------------------------------------------------------
    def _vols(self, V, Cv, Sv):
        assert V.dtype == np.uint32 and V.flags.c_contiguous and V.shape == self.shape
        assert Cv.dtype == np.uint8 and Cv.flags.c_contiguous and Cv.shape == self.shape
        if Sv is not None:
            assert Sv.dtype == np.uint8 and Sv.flags.c_contiguous and Sv.shape == self.shape

    def sweep(self, m, V, Cv, Sv=None):
        self._vols(V, Cv, Sv)
        _load().orc_sweep(self._h, m, _ptr(V), _ptr(Cv), _ptr(Sv))

    def cycles(self, V, Cv, Sv, ncycles):
        self._vols(V, Cv, Sv)
        _load().orc_cycles(self._h, _ptr(V), _ptr(Cv), _ptr(Sv), ncycles)

    def run(self, Cv, Sv, start, ncycles):
        V = np.empty(self.shape, np.uint32)
        self._vols(V, Cv, Sv)
        rc = _load().orc_run(self._h, _ptr(V), _ptr(Cv), _ptr(Sv), start[0], start[1], start[2], ncycles)
        if rc:
            raise OracleError(rc, "run")
        return V

    def run_from(self, Cv, Sv, start, m0, ncycles):
        """N-turn run with maneuver m0 in progress at the start (DESIGN R26); m0 = -1: plain run."""
        V = np.empty(self.shape, np.uint32)
        self._vols(V, Cv, Sv)
        L = _load()
        L.orc_run_from.argtypes = [C.c_void_p] + [C.c_void_p] * 3 + [C.c_int] * 5
        rc = L.orc_run_from(self._h, _ptr(V), _ptr(Cv), _ptr(Sv), start[0], start[1], start[2], int(m0), ncycles)
        if rc:
            raise OracleError(rc, "run_from")
        return V

    def backtrack_from(self, V, Cv, Sv, start, m0, goal, cap=4096):
        self._vols(V, Cv, Sv)
        out = (_Waypoint * cap)()
        cnt, cost = C.c_int(0), C.c_uint32(0)
        L = _load()
        L.orc_backtrack_from.argtypes = [C.c_void_p] + [C.c_void_p] * 3 + [C.c_int] * 7 + [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        rc = L.orc_backtrack_from(self._h, _ptr(V), _ptr(Cv), _ptr(Sv), start[0], start[1], start[2], int(m0),
                                  goal[0], goal[1], goal[2], out, cap, C.byref(cnt), C.byref(cost))
        if rc:
            raise OracleError(rc, "backtrack")
        return [(w.i, w.j, w.theta, w.m) for w in out[:cnt.value]], cost.value

    def dijkstra(self, Cv, Sv, start, kind="star", m0=-1):
        V = np.empty(self.shape, np.uint32)
        self._vols(V, Cv, Sv)
        L = _load()
        L.orc_dijkstra_from.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        rc = L.orc_dijkstra_from(self._h, 0 if kind == "star" else 1, _ptr(Cv), _ptr(Sv), start[0], start[1], start[2], int(m0), _ptr(V))
        if rc:
            raise OracleError(rc, "dijkstra")
        return V

    def graph_size_at(self, Cv, Sv, start, cell, kind="star"):
        """(vertices settled, edges relaxed) at `cell` = (i, j, theta) by one Dijkstra run: k_V, k_E of Table 1."""
        L = _load()
        L.orc_dijkstra_probe.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.orc_dijkstra_probe_result.argtypes = [C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.orc_dijkstra_probe(self._h, cell[0], cell[1], cell[2])
        try:
            self.dijkstra(Cv, Sv, start, kind)
            kv, ke = C.c_int(0), C.c_int(0)
            L.orc_dijkstra_probe_result(C.byref(kv), C.byref(ke))
        finally:
            L.orc_dijkstra_probe(self._h, -1, -1, -1)
        return kv.value, ke.value

    def backtrack(self, V, Cv, Sv, start, goal, cap=4096):
        self._vols(V, Cv, Sv)
        out = (_Waypoint * cap)()
        cnt, cost = C.c_int(0), C.c_uint32(0)
        rc = _load().orc_backtrack(self._h, _ptr(V), _ptr(Cv), _ptr(Sv), start[0], start[1], start[2],
                                   goal[0], goal[1], goal[2], out, cap, C.byref(cnt), C.byref(cost))
        if rc:
            raise OracleError(rc, "backtrack")
        return [(w.i, w.j, w.theta, w.m) for w in out[:cnt.value]], cost.value

    def reach_run(self, Cv, start, n_levels):
        """Appendix C: K[X] = fewest maneuvers that reach X (255 = more than n_levels), uint8."""
        K = np.empty(self.shape, np.uint8)
        L = _load()
        L.orc_reach_run.restype = C.c_int
        L.orc_reach_run.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]
        assert Cv.dtype == np.uint8 and Cv.flags.c_contiguous and Cv.shape == self.shape
        rc = L.orc_reach_run(self._h, _ptr(K), _ptr(Cv), start[0], start[1], start[2], int(n_levels))
        if rc:
            raise OracleError(rc, "reach_run")
        return K

    def reach_backtrack(self, K, Cv, start, goal, cap=4096):
        out = (_Waypoint * cap)()
        cnt, cost = C.c_int(0), C.c_uint32(0)
        L = _load()
        L.orc_reach_backtrack.restype = C.c_int
        L.orc_reach_backtrack.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p] + [C.c_int] * 6 + [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        rc = L.orc_reach_backtrack(self._h, _ptr(K), _ptr(Cv), start[0], start[1], start[2], goal[0], goal[1], goal[2],
                                   out, cap, C.byref(cnt), C.byref(cost))
        if rc:
            raise OracleError(rc, "reach_backtrack")
        return [(w.i, w.j, w.theta, w.m) for w in out[:cnt.value]], cost.value

    def goal_search(self, V, goals, d, W, w):
        """Section IX under reading DESIGN R20: best vertex of the goal sets of `goals`
        (list of (i, j, theta)) by V + W (di^2 + dj^2) + w dt^2.  Returns ((i, j, theta), goal index, score)."""
        L = _load()
        L.orc_goal_search.restype = C.c_int
        L.orc_goal_search.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_uint32, C.c_uint32,
                                      C.c_void_p, C.POINTER(C.c_uint64)]
        g = np.ascontiguousarray(np.asarray(goals, np.int32).reshape(-1, 3))
        out = np.zeros(4, np.int32)
        score = C.c_uint64(0)
        assert V.dtype == np.uint32 and V.flags.c_contiguous and V.shape == self.shape
        rc = L.orc_goal_search(self._h, _ptr(V), g.ctypes.data_as(C.c_void_p), len(g), int(d), int(W), int(w),
                               out.ctypes.data_as(C.c_void_p), C.byref(score))
        if rc:
            raise OracleError(rc, "goal_search")
        return (int(out[0]), int(out[1]), int(out[2])), int(out[3]), int(score.value)


def soft_from_hard(hard: np.ndarray, k: float = 4.0):
    """Steps 1-2 of PAPER.md:388-389 under reading DESIGN R17: exact squared distance transform of hard | wall,
    float32 distance, Q4.4 soft image.  Returns (d2 int32, dist float32, soft uint8)."""
    L = _load_dt()
    h = np.ascontiguousarray(hard, np.uint8)
    n = h.shape[0]
    d2 = np.empty((n, n), np.int32); dist = np.empty((n, n), np.float32); soft = np.empty((n, n), np.uint8)
    rc = L.orc_soft_from_hard(h.ctypes.data_as(C.c_void_p), n, C.c_float(k), d2.ctypes.data_as(C.c_void_p),
                              dist.ctypes.data_as(C.c_void_p), soft.ctypes.data_as(C.c_void_p))
    assert rc == 0
    return d2, dist, soft


def edt_brute(hard: np.ndarray) -> np.ndarray:
    """Squared distance to the nearest pixel of hard | wall by the O(N^4) definition (tiny images only)."""
    L = _load_dt()
    h = np.ascontiguousarray(hard, np.uint8)
    n = h.shape[0]
    d2 = np.empty((n, n), np.int32)
    L.orc_edt_brute(h.ctypes.data_as(C.c_void_p), n, d2.ctypes.data_as(C.c_void_p))
    return d2


def _load_dt():
    build()
    L = C.CDLL(_LIB)
    L.orc_soft_from_hard.restype = C.c_int
    L.orc_soft_from_hard.argtypes = [C.c_void_p, C.c_int, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
    L.orc_edt_brute.restype = None
    L.orc_edt_brute.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
    return L
