"""ctypes binding with the same names as the C ABI (include/nhplan.h)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libnhplan.so")

INF = 0xFFFFFFFF
FLAG_FORWARD_ONLY, FLAG_SOFT, FLAG_SIMPLE_KERNELS, FLAG_FIXED_WORK, FLAG_NO_SHORTCUTS, FLAG_SECTIONS, FLAG_NO_SECTIONS = 1, 2, 4, 8, 16, 32, 64
DEFAULT_CYCLES = 8                                          # NHP_DEFAULT_CYCLES
PLAN_EAGER = 128                                            # waypoints that come back with the status words (NHP_PLAN_EAGER)
MANEUVER_NAMES = ("LF", "SF", "RB", "RF", "SB", "LB")
ERRORS = {-1: "NHP_E_ARG", -2: "NHP_E_NOT_POW2", -3: "NHP_E_ANGRES", -4: "NHP_E_START_BLOCKED",
          -5: "NHP_E_GOAL_UNREACHED", -6: "NHP_E_BUFFER", -7: "NHP_E_CUDA", -8: "NHP_E_STATE", -9: "NHP_E_WEIGHTS"}

EXPORTS = ("nhp_query_sizes", "nhp_planner_create", "nhp_planner_destroy", "nhp_last_error",
           "nhp_render_vehicle_footprint", "nhp_set_box", "nhp_render_obstacles", "nhp_render_obstacles_dt", "nhp_debug_soft_image",
           "nhp_run_nturn", "nhp_run_nturn_from", "nhp_reach_run", "nhp_reach_levels", "nhp_reach_count_volume", "nhp_reach_extract_path", "nhp_run_more",
           "nhp_cost_volume", "nhp_extract_path", "nhp_extract_path_goalset", "nhp_status", "nhp_index_to_pose", "nhp_pose_to_index",
           "nhp_debug_tables", "nhp_debug_footprint", "nhp_launch_count", "nhp_set_profiling", "nhp_kernel_times", "nhp_prof_dropped", "nhp_microbench_alu", "nhp_microbench_read",
           "nhp_soft_from_hard_noalloc", "nhp_noalloc_last_error", "nhp_debug_set_plan_eager", "nhp_debug_cycle_graph_kernels", "nhp_set_lane_penalty")
KERNEL_SLOTS = 17
KERNEL_SLOT_NAMES = ("LF", "SF", "RB", "RF", "SB", "LB", "render_collision", "render_soft", "init_export",
                     "backtrack", "raster_pack", "turn_pair", "distance_transform", "reach_level", "straight_xrows", "straight_rows", "straight_sect")
NESTED_SLOTS = ("straight_xrows", "straight_rows", "straight_sect")        # bracketed inside SF / SB: not part of a sum over the slots


class Weights(C.Structure):
    _fields_ = [("ct", C.c_uint32 * 6), ("dir_mult", C.c_uint32 * 6), ("cost_one_log2", C.c_int32), ("flags", C.c_int32)]


class Sizes(C.Structure):
    _fields_ = [("V_bytes", C.c_size_t), ("C_bytes", C.c_size_t), ("S_bytes", C.c_size_t), ("workspace_bytes", C.c_size_t)]


class Limits(C.Structure):
    _fields_ = [("max_footprint_radius", C.c_int32), ("max_reach_levels", C.c_int32)]


class Buffers(C.Structure):
    _fields_ = [("V", C.c_void_p), ("C", C.c_void_p), ("S", C.c_void_p), ("workspace", C.c_void_p)]


class Waypoint(C.Structure):
    _fields_ = [("i", C.c_int32), ("j", C.c_int32), ("theta", C.c_int32), ("m", C.c_int32)]


class NhpError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


_lib = None


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen libnhplan.so; fails loudly if it has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2306_01301_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(_LIB_PATH)
        L.nhp_query_sizes.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(Limits), C.POINTER(Sizes)]
        L.nhp_planner_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_double, C.POINTER(Weights),
                                         C.POINTER(Limits), C.POINTER(Buffers), C.c_void_p]
        L.nhp_planner_destroy.argtypes = [C.c_void_p]
        L.nhp_last_error.argtypes = [C.c_void_p]
        L.nhp_last_error.restype = C.c_char_p
        L.nhp_render_vehicle_footprint.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double]
        L.nhp_set_box.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.nhp_render_obstacles.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.nhp_render_obstacles_dt.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_void_p]
        L.nhp_debug_soft_image.argtypes = [C.c_void_p, C.c_void_p]
        L.nhp_set_lane_penalty.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.nhp_debug_set_plan_eager.argtypes = [C.c_void_p, C.c_int]
        L.nhp_debug_cycle_graph_kernels.argtypes = [C.c_void_p]
        L.nhp_run_nturn.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]
        L.nhp_run_nturn_from.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
        L.nhp_reach_run.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]
        L.nhp_reach_levels.argtypes = [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_int)]
        L.nhp_reach_count_volume.argtypes = [C.c_void_p, C.c_void_p]
        L.nhp_reach_extract_path.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.POINTER(Waypoint), C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.nhp_run_more.argtypes = [C.c_void_p, C.c_int]
        L.nhp_cost_volume.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
        L.nhp_extract_path.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.POINTER(Waypoint), C.c_int,
                                       C.POINTER(C.c_int), C.POINTER(C.c_uint32)]
        L.nhp_extract_path_goalset.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_uint32, C.c_uint32, C.POINTER(Waypoint),
                                               C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_uint32), C.c_void_p, C.POINTER(C.c_uint64)]
        L.nhp_status.argtypes = [C.c_void_p]
        L.nhp_index_to_pose.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int] + [C.POINTER(C.c_double)] * 3
        L.nhp_pose_to_index.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double] + [C.POINTER(C.c_int)] * 3
        L.nhp_debug_tables.argtypes = [C.c_void_p] + [C.c_void_p] * 6
        L.nhp_debug_footprint.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.c_void_p, C.c_size_t]
        L.nhp_prof_dropped.argtypes = [C.c_void_p]
        L.nhp_prof_dropped.restype = C.c_longlong
        L.nhp_launch_count.argtypes = [C.c_void_p]
        L.nhp_launch_count.restype = C.c_longlong
        L.nhp_set_profiling.argtypes = [C.c_void_p, C.c_int]
        L.nhp_kernel_times.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_longlong), C.c_int]
        L.nhp_microbench_alu.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int)]
        L.nhp_microbench_read.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double)]
        L.nhp_soft_from_hard_noalloc.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nhp_noalloc_last_error.argtypes = []
        L.nhp_noalloc_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def query_sizes(log2_n, log2_ntheta, flags=0, max_footprint_radius=0, max_reach_levels=0):
    s = Sizes()
    lim = Limits(max_footprint_radius, max_reach_levels)
    rc = load_library().nhp_query_sizes(log2_n, log2_ntheta, flags, C.byref(lim), C.byref(s))
    if rc:
        raise NhpError(rc, "query_sizes")
    return s


NOALLOC_MAX_N = 1024                                        # NHP_NOALLOC_MAX_N


def soft_from_hard_noalloc(hard, k, soft_out, dist_out=None, stream=None):
    """nhp_soft_from_hard_noalloc: distance transform + soft image of an n x n obstacle image, n <= NOALLOC_MAX_N, without a
    planner handle and without any allocation inside the library -- for callers that may not allocate device memory after
    start-up (control loops with a fixed memory budget, guests of a process whose pool already owns the GPU's memory).
    The caller brings every buffer: `hard` (uint8, n x n), `soft_out` (uint8, n x n) and optionally `dist_out` (float32,
    n x n), all contiguous CUDA tensors on one device; `stream` is a torch stream of that device (default: its current one).
    The work is enqueued, not waited for.  All calls on a device share one built-in scratch image: calls that could overlap on
    the GPU must be ordered by the caller (include/nhplan.h has the full contract)."""
    import torch
    L = load_library()
    n = hard.shape[0]
    for t, dt in ((hard, torch.uint8), (soft_out, torch.uint8), (dist_out, torch.float32)):
        if t is not None:
            assert t.is_cuda and t.dtype == dt and t.is_contiguous() and tuple(t.shape) == (n, n)
    st = stream if stream is not None else torch.cuda.current_stream(hard.device)
    rc = L.nhp_soft_from_hard_noalloc(hard.data_ptr(), int(n), float(k), soft_out.data_ptr(),
                                      dist_out.data_ptr() if dist_out is not None else None, C.c_void_p(st.cuda_stream))
    if rc:
        raise NhpError(rc, f"soft_from_hard_noalloc: {L.nhp_noalloc_last_error().decode()}")


class Planner:
    """One planner handle = one grid, one stream.  Method names follow the C ABI without the nhp_ prefix."""

    GUARD_BYTE = 0xA5

    def __init__(self, log2_n, log2_ntheta, R, ct, dir_mult=(256,) * 6, cost_one_log2=10, flags=0, device="cuda:0",
                 stream=None, max_footprint_radius=0, reach_levels=0, guard_bytes=0):
        """max_footprint_radius / reach_levels: the nhp_limits the workspace is sized for (0 = the library's defaults:
        radius min(64, N/2 - 1), no reachability planner).  guard_bytes > 0 (a multiple of 256; test aid): every buffer
        handed to the library sits between two guard bands of that many bytes, see guards_intact()."""
        import torch
        self._L = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2306_01301_b200.Planner needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.n, self.nt = 1 << log2_n, 1 << log2_ntheta
        self.shape = (self.nt, self.n, self.n)
        self.flags = flags
        sz = query_sizes(log2_n, log2_ntheta, flags, max_footprint_radius, reach_levels)
        assert guard_bytes % 256 == 0
        self._guarded = []

        def buf(nbytes, dtype):
            raw = torch.empty(nbytes + 2 * guard_bytes, dtype=torch.uint8, device=self.device)
            if guard_bytes:
                raw[:guard_bytes] = self.GUARD_BYTE
                raw[guard_bytes + nbytes:] = self.GUARD_BYTE
                self._guarded.append((raw, nbytes))
            return raw[guard_bytes:guard_bytes + nbytes].view(dtype)

        with torch.cuda.device(self.device):
            self.V = buf(sz.V_bytes, torch.int32)
            self.C = buf(sz.C_bytes, torch.int32)
            self.S = buf(sz.S_bytes, torch.uint8) if sz.S_bytes else None
            self.W = buf(sz.workspace_bytes, torch.uint8)
            self._guard_bytes = guard_bytes
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            w = Weights((C.c_uint32 * 6)(*ct), (C.c_uint32 * 6)(*dir_mult), cost_one_log2, flags)
            b = Buffers(self.V.data_ptr(), self.C.data_ptr(), self.S.data_ptr() if self.S is not None else None, self.W.data_ptr())
            lim = Limits(max_footprint_radius, reach_levels)
            h = C.c_void_p()
            rc = self._L.nhp_planner_create(C.byref(h), log2_n, log2_ntheta, float(R), C.byref(w), C.byref(lim), C.byref(b),
                                            C.c_void_p(self.stream.cuda_stream))
        if rc:
            raise NhpError(rc, "planner_create")
        self._h = h

    def guards_intact(self):
        """True iff no byte of any guard band around V, C, S and the workspace has been written (needs guard_bytes > 0)."""
        self.torch.cuda.synchronize(self.device)
        g = self._guard_bytes
        return all(bool((raw[:g] == self.GUARD_BYTE).all()) and bool((raw[g + n:] == self.GUARD_BYTE).all()) for raw, n in self._guarded)

    @classmethod
    def from_scene(cls, sc, flags=0, **kw):
        f = flags | sc.flags | (FLAG_SOFT if sc.soft is not None else 0)
        p = cls(sc.log2_n, sc.log2_nt, sc.R, sc.ct, sc.dir_mult, sc.cost_one_log2, f, **kw)
        p.render_vehicle_footprint(sc.mask, sc.ou, sc.ov)
        return p

    def close(self):
        if getattr(self, "_h", None):
            self._L.nhp_planner_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        if rc:
            raise NhpError(rc, f"{what}: {self._L.nhp_last_error(self._h).decode()}")

    # ---- the ABI calls ---------------------------------------------------------------------
    def render_vehicle_footprint(self, mask, origin_u, origin_v):
        mask = np.ascontiguousarray(mask, np.uint8)
        self._check(self._L.nhp_render_vehicle_footprint(self._h, mask.ctypes.data, mask.shape[1], mask.shape[0],
                                                         float(origin_u), float(origin_v)), "render_vehicle_footprint")

    def set_box(self, f, r, s):
        """Bounding-box vehicle of appendix G: u in [-r, f), v in [-s, s) cells around the rear axle."""
        self._check(self._L.nhp_set_box(self._h, int(f), int(r), int(s)), "set_box")

    def render_obstacles(self, hard, soft=None):
        """hard / soft: numpy uint8 arrays or CPU torch tensors (host path, copied inside the call) or CUDA tensors."""
        def ptr(a):
            if a is None:
                return None, 0
            if isinstance(a, np.ndarray):
                assert a.dtype == np.uint8 and a.flags.c_contiguous and a.shape == (self.n, self.n)
                return a.ctypes.data, 0
            assert a.dtype == self.torch.uint8 and a.is_contiguous() and tuple(a.shape) == (self.n, self.n)
            return a.data_ptr(), int(a.is_cuda)
        hp, hd = ptr(hard)
        sp, sd = ptr(soft)
        assert soft is None or hd == sd
        self._keep = (hard, soft)                       # host buffers must outlive the async copy
        self._check(self._L.nhp_render_obstacles(self._h, hp, sp, hd), "render_obstacles")

    def set_lane_penalty(self, lane_dir=None, lane_pen=None):
        """Lane map of nhp_set_lane_penalty (area / orientation penalty, DESIGN R28): two (N, N) uint8 images, numpy (host path)
        or CUDA tensors; None, None switches it off.  Takes effect at the next render_obstacles / render_obstacles_dt."""
        if lane_dir is None and lane_pen is None:
            self._check(self._L.nhp_set_lane_penalty(self._h, None, None, 0), "set_lane_penalty")
            return
        ptrs, dev = [], []
        for a in (lane_dir, lane_pen):
            if isinstance(a, np.ndarray):
                assert a.dtype == np.uint8 and a.flags.c_contiguous and a.shape == (self.n, self.n)
                ptrs.append(a.ctypes.data); dev.append(0)
            else:
                assert a.dtype == self.torch.uint8 and a.is_contiguous() and tuple(a.shape) == (self.n, self.n)
                ptrs.append(a.data_ptr()); dev.append(int(a.is_cuda))
        assert dev[0] == dev[1]
        self._keep_lane = (lane_dir, lane_pen)             # host buffers must outlive the async copy
        self._check(self._L.nhp_set_lane_penalty(self._h, ptrs[0], ptrs[1], dev[0]), "set_lane_penalty")

    def render_obstacles_dt(self, hard, k=4.0, dist_out=None):
        """Distance transform + soft image on the device, then rendering (nhp_render_obstacles_dt).
        dist_out: optional float32 CUDA tensor (N, N) that receives the distance image."""
        if isinstance(hard, np.ndarray):
            assert hard.dtype == np.uint8 and hard.flags.c_contiguous and hard.shape == (self.n, self.n)
            hp, hd = hard.ctypes.data, 0
        else:
            assert hard.dtype == self.torch.uint8 and hard.is_contiguous() and tuple(hard.shape) == (self.n, self.n)
            hp, hd = hard.data_ptr(), int(hard.is_cuda)
        dp = None
        if dist_out is not None:
            assert dist_out.is_cuda and dist_out.dtype == self.torch.float32 and dist_out.is_contiguous()
            assert tuple(dist_out.shape) == (self.n, self.n)
            dp = dist_out.data_ptr()
        self._keep = (hard, dist_out)
        self._check(self._L.nhp_render_obstacles_dt(self._h, hp, hd, float(k), dp), "render_obstacles_dt")

    def soft_image_numpy(self):
        out = np.empty((self.n, self.n), np.uint8)
        self._check(self._L.nhp_debug_soft_image(self._h, out.ctypes.data), "debug_soft_image")
        return out

    def run_nturn(self, start, n_cycles=DEFAULT_CYCLES):
        self._check(self._L.nhp_run_nturn(self._h, int(start[0]), int(start[1]), int(start[2]), int(n_cycles)), "run_nturn")

    def cycle_graph_kernels(self):
        """Kernels in the CUDA graph of one inner cycle that run_nturn replays while profiling is off; 0 = separate launches."""
        return int(self._L.nhp_debug_cycle_graph_kernels(self._h))

    def debug_set_plan_eager(self, n_waypoints):
        """Waypoints that come back with the status words (test aid: a small number exercises the second copy)."""
        self._check(self._L.nhp_debug_set_plan_eager(self._h, int(n_waypoints)), "debug_set_plan_eager")

    def run_nturn_from(self, start, m0, n_cycles=DEFAULT_CYCLES):
        """run_nturn with maneuver m0 (0..5 in cycle order, -1 = none) in progress at the start."""
        self._check(self._L.nhp_run_nturn_from(self._h, int(start[0]), int(start[1]), int(start[2]), int(m0), int(n_cycles)),
                    "run_nturn_from")

    def reach_run(self, start, n_levels=8):
        """Reachability (bit-vector) planner of appendix C: level volumes 0 .. n_levels from `start`."""
        self._check(self._L.nhp_reach_run(self._h, int(start[0]), int(start[1]), int(start[2]), int(n_levels)), "reach_run")

    def reach_count_numpy(self):
        """K[theta, j, i] = fewest maneuvers that reach the pose (255 = not within the levels of the last reach_run)."""
        K = self.torch.empty(self.shape, dtype=self.torch.uint8, device=self.device)
        self._check(self._L.nhp_reach_count_volume(self._h, K.data_ptr()), "reach_count_volume")
        return K.cpu().numpy()

    def reach_extract_path(self, goal, cap=4096):
        buf = (Waypoint * cap)()
        cnt, nm = C.c_int(0), C.c_int(0)
        self._check(self._L.nhp_reach_extract_path(self._h, int(goal[0]), int(goal[1]), int(goal[2]), buf, cap,
                                                   C.byref(cnt), C.byref(nm)), "reach_extract_path")
        return [(w.i, w.j, w.theta, w.m) for w in buf[:cnt.value]], nm.value

    def run_more(self, n_cycles):
        self._check(self._L.nhp_run_more(self._h, int(n_cycles)), "run_more")

    def cost_volume(self):
        """Canonical cost-to-come volume as a (N_theta, N, N) int32 CUDA tensor view of V (bit pattern = uint32)."""
        out = C.c_void_p()
        self._check(self._L.nhp_cost_volume(self._h, C.byref(out)), "cost_volume")
        assert out.value == self.V.data_ptr()
        return self.V.view(self.shape)

    def extract_path(self, goal, cap=4096):
        buf = (Waypoint * cap)()
        cnt, cost = C.c_int(0), C.c_uint32(0)
        self._check(self._L.nhp_extract_path(self._h, int(goal[0]), int(goal[1]), int(goal[2]), buf, cap,
                                             C.byref(cnt), C.byref(cost)), "extract_path")
        return [(w.i, w.j, w.theta, w.m) for w in buf[:cnt.value]], cost.value

    def extract_path_goalset(self, goals, d, W, w, cap=4096):
        """Goal search over the goal sets of `goals` (list of (i, j, theta)) + back-tracking from the winner.
        Returns (plan, cost, (i, j, theta), goal index, score)."""
        g = np.ascontiguousarray(np.asarray(goals, np.int32).reshape(-1, 3))
        buf = (Waypoint * cap)()
        cnt, cost, score = C.c_int(0), C.c_uint32(0), C.c_uint64(0)
        chosen = np.zeros(4, np.int32)
        self._check(self._L.nhp_extract_path_goalset(self._h, g.ctypes.data, len(g), int(d), int(W), int(w), buf, cap,
                                                     C.byref(cnt), C.byref(cost), chosen.ctypes.data, C.byref(score)),
                    "extract_path_goalset")
        return ([(x.i, x.j, x.theta, x.m) for x in buf[:cnt.value]], cost.value,
                (int(chosen[0]), int(chosen[1]), int(chosen[2])), int(chosen[3]), int(score.value))

    def status(self):
        self._check(self._L.nhp_status(self._h), "status")

    def index_to_pose(self, i, j, theta):
        x, y, t = C.c_double(), C.c_double(), C.c_double()
        self._check(self._L.nhp_index_to_pose(self._h, i, j, theta, C.byref(x), C.byref(y), C.byref(t)), "index_to_pose")
        return x.value, y.value, t.value

    def pose_to_index(self, x, y, theta_rad):
        i, j, t = C.c_int(), C.c_int(), C.c_int()
        self._check(self._L.nhp_pose_to_index(self._h, x, y, theta_rad, C.byref(i), C.byref(j), C.byref(t)), "pose_to_index")
        return i.value, j.value, t.value

    def debug_tables(self):
        n, nt = self.n, self.nt
        t = dict(beta=np.empty(nt, np.int32), psi2=np.empty(nt, np.uint8), B=np.empty((nt, n), np.int32),
                 I=np.empty(nt, np.uint8), J=np.empty(nt, np.int8), len_q=np.empty((6, nt), np.uint32))
        self._check(self._L.nhp_debug_tables(self._h, *[t[k].ctypes.data for k in ("beta", "psi2", "B", "I", "J", "len_q")]),
                    "debug_tables")
        return t

    def debug_footprint(self):
        """E_Theta of the current footprint: (rad, covered uint8 [N_theta][2 rad + 1][2 rad + 1])."""
        rad = C.c_int(0)
        self._check(self._L.nhp_debug_footprint(self._h, C.byref(rad), None, 0), "debug_footprint")
        side = 2 * rad.value + 1
        cov = np.empty((self.nt, side, side), np.uint8)
        self._check(self._L.nhp_debug_footprint(self._h, C.byref(rad), cov.ctypes.data, cov.nbytes), "debug_footprint")
        return rad.value, cov

    def prof_dropped(self):
        return int(self._L.nhp_prof_dropped(self._h))

    def microbench_alu(self, chains=8):
        """-> (VIADDMNMX lane-operations per second, SM count): the integer-pipe peak of DESIGN.md section 6.7, measured."""
        ops, sms = C.c_double(0), C.c_int(0)
        self._check(self._L.nhp_microbench_alu(self._h, int(chains), C.byref(ops), C.byref(sms)), "microbench_alu")
        return ops.value, sms.value

    def microbench_read(self, pattern):
        """-> bytes per second of a pure read of V in the access pattern of a sweep kernel (0 linear, 1 rows, 2 x-rows, 3 turn tiles)."""
        bps = C.c_double(0)
        self._check(self._L.nhp_microbench_read(self._h, int(pattern), C.byref(bps)), "microbench_read")
        return bps.value

    def launch_count(self):
        return int(self._L.nhp_launch_count(self._h))

    def set_profiling(self, enable=True):
        self._check(self._L.nhp_set_profiling(self._h, int(bool(enable))), "set_profiling")

    def kernel_times(self, reset=False):
        """-> {slot name: (summed ms, launches)} of the event-bracketed launches since the last reset."""
        ms = (C.c_double * KERNEL_SLOTS)()
        cnt = (C.c_longlong * KERNEL_SLOTS)()
        self._check(self._L.nhp_kernel_times(self._h, ms, cnt, int(bool(reset))), "kernel_times")
        return {KERNEL_SLOT_NAMES[k]: (ms[k], cnt[k]) for k in range(KERNEL_SLOTS)}

    # ---- host copies for tests ---------------------------------------------------------------
    def cost_volume_numpy(self):
        return self.cost_volume().cpu().numpy().view(np.uint32)

    def collision_numpy(self):
        """Unpacked collision volume, uint8 {0,1} [Theta][j][i]."""
        words = self.C.cpu().numpy().view(np.uint32)
        bits = np.unpackbits(words.view(np.uint8), bitorder="little")
        return bits.reshape(self.shape)

    def soft_numpy(self):
        return None if self.S is None else self.S.cpu().numpy().reshape(self.shape)
