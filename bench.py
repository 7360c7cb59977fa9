"""bench.py -- one JSON line for the N-turn planner hot path on B200 (contract: see DESIGN.md section 9).

A "step" is one pass of the whole hot path over one synthetic scene:
    render_obstacles (collision [+ soft] volume)  ->  run_nturn (N_T maneuver cycles)  ->  extract_path
`value`  = pose-updates / s with the obstacle images already resident in HBM (6 * N_T * N_R pose-updates per plan,
           PAPER.md:453), whole job over all ranks (replicas only: one independent plan per GPU, no collective);
`e2e`    = the same metric through the public API with HOST (pinned) obstacle images: the H2D copy of the images
           and the D2H copy of the plan are inside the timed region;
`roofline` = the dominant kernel's algorithmic bytes / its average CUDA-event duration over the timed region,
           against the measured HBM copy bandwidth in MEASURED_PEAKS.json;
`cpu_baseline` = the CPU oracle, as it stands, on a bounded sample of the same workload on this box's host cores.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pose_updates_per_sec (N-turn planner, whole plan: render + N_T maneuver cycles + back-track)"   # ours; the reference arm
# times maneuver sweeps of the oracle over the same volume (its `sample` says which) and reports them in the same unit
UNIT = "Gpose-updates/s"
FALLBACK_HBM_GBS = 6650.0            # /opt/skills/guides/B200_PROFILING.md fallback
ALG_BYTES_HARD, ALG_BYTES_SOFT = 8.125, 9.125     # read V 4 + write V 4 + 1 collision bit [+ 1 soft byte]


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs[k-1]; 3 = 512^3 maze (default)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cycles", type=int, default=0, help="override N_T (0 = the config's own)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--simple-kernels", action="store_true", help="thread-per-curve bring-up kernels (A/B)")
    ap.add_argument("--reach", action="store_true",
                    help="time the reachability (bit-vector) planner of appendix C instead: render + N_T levels + back-track")
    ap.add_argument("--fixed-work", action="store_true", help="NHP_FLAG_FIXED_WORK: data-dependent short cuts off (PAPER.md:565)")
    ap.add_argument("--no-shortcuts", action="store_true", help="NHP_FLAG_NO_SHORTCUTS: every warp runs every pass; stores still only where a value improved")
    ap.add_argument("--sections", action="store_true", help="NHP_FLAG_SECTIONS: straight sweeps by Sections (appendix D) also at 512 cells per side")
    ap.add_argument("--no-sections", action="store_true", help="NHP_FLAG_NO_SECTIONS: streaming straight kernels also on small grids")
    ap.add_argument("--no-extra", action="store_true", help="skip the fixed-work pass and the configs 4 / 5 side runs")
    ap.add_argument("--dt-on-device", action="store_true",
                    help="soft configs: distance transform + soft image on the GPU (nhp_render_obstacles_dt) instead of the harness image")
    return ap.parse_args()


def workload_name(sc, n_cycles):
    return (f"{sc.name}: {sc.n}x{sc.n}x{sc.nt} (x,y,theta), vehicle {sc.mask.shape[1]}x{sc.mask.shape[0]}, R={sc.R:g}, "
            f"N_T={n_cycles}, {'soft+hard' if sc.soft is not None else 'hard'} obstacles")


SLOT_SOURCES = {"straight_xrows": "straight.cu", "straight_rows": "straight.cu", "straight_sect": "straight.cu", "SF": "straight.cu", "SB": "straight.cu",
                "render_collision": "render.cu", "render_soft": "render.cu", "backtrack": "backtrack.cu", "distance_transform": "distance.cu"}     # default: sweep.cu


def source_hashes():
    """sha256 (first 16 hex digits) of every kernel source: a committed ncu byte count is only divided by a fresh time when the
    kernel's source (and the shared header) is still the one the capture was taken from."""
    import glob
    import hashlib
    d = os.path.join(ROOT, "paper_2306_01301_b200", "csrc")
    return {os.path.basename(p): hashlib.sha256(open(p, "rb").read()).hexdigest()[:16] for p in sorted(glob.glob(os.path.join(d, "*.cu*")))}


def traffic_table():
    """profiles/traffic.csv -> ({(config, slot): (bytes, source)}, {file: sha16 at capture}, commit the captures were taken at)."""
    rows, hashes, commit = {}, {}, None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for ln in f:
                ln = ln.strip()
                if ln.startswith("# sha16 "):
                    hashes = dict(kv.split("=") for kv in ln[8:].split())
                elif ln.startswith("# commit "):
                    commit = ln[9:].strip()
                elif ln and not ln.startswith("#"):
                    c, k, b, src = ln.split(",", 3)
                    rows[(c, k)] = (int(b), src)
    except OSError:
        pass
    return rows, hashes, commit


def measured_traffic(config, slot):
    """dram bytes per launch of `slot` from the committed ncu capture (profiles/traffic.csv), or None.  `stale` = the kernel's
    source or the shared header changed since the capture: the bytes are shown, frac_traffic is not computed from them."""
    rows, hashes, _ = traffic_table()
    if (str(config), slot) not in rows:
        return None
    now = source_hashes()
    files = (SLOT_SOURCES.get(slot, "sweep.cu"), "nhp_internal.cuh")
    b, src = rows[(str(config), slot)]
    return {"bytes_per_launch": b, "source": src, "stale": any(hashes.get(fn) != now.get(fn) for fn in files)}


def peak_hbm():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.th = threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.th.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def bench_config(sc, n_cycles, args, ws, dt_dev=False):
    """The `config` object of the JSON line: the workload and how it is run, the same keys for both arms."""
    n_r = sc.n * sc.n * sc.nt
    return {"workload": workload_name(sc, n_cycles), "baseline_config": args.config, "pose_updates_per_plan": 6 * n_cycles * n_r,
            "parallelism": f"replicas x{ws} (no collective)",
            "soft_image": ("device distance transform" if dt_dev else "harness (CPU)") if sc.soft is not None else None,
            "l2": f"inputs larger than L2: value volume {4 * n_r / 2**20:.0f} MiB vs 126 MB L2, every sweep streams it",
            "fixed_work": bool(args.fixed_work), "no_shortcuts": bool(args.no_shortcuts)}


def pick_goal(p, sc, torch):
    """The nominal goal if the sweeps reached it, else the reached candidate of largest finite cost
    (N_T cycles only guarantee plans of <= N_T maneuvers).  Harness logic on <= 257 values."""
    cands = [sc.goal] + list(sc.extra_goals)
    V = p.cost_volume()
    idx = torch.tensor([(t * sc.n + j) * sc.n + i for (i, j, t) in cands], device=V.device)
    vals = V.view(-1)[idx].to(torch.int64) & 0xFFFFFFFF
    vals = vals.cpu().tolist()
    if vals[0] != 0xFFFFFFFF:
        return tuple(sc.goal)
    best = max(range(len(cands)), key=lambda k: (-1 if vals[k] == 0xFFFFFFFF else vals[k]))
    return tuple(cands[best]) if vals[best] != 0xFFFFFFFF else tuple(sc.start)


SWEEP_SLOTS = ("turn_pair", "LF", "RB", "RF", "LB", "straight_xrows", "straight_rows", "straight_sect")


class PlanBench:
    """One planner on one scene: warm-up, goal choice, and timed passes of `step` = render + N_T cycles + back-track."""

    def __init__(self, nhp, torch, replicas, sc, n_cycles, dev, flags=0, reach=False, dt_on_device=False):
        self.nhp, self.torch, self.replicas, self.sc, self.n_cycles, self.dev = nhp, torch, replicas, sc, n_cycles, dev
        self.reach, self.dt_dev = reach, dt_on_device and sc.soft is not None
        self.p = nhp.Planner.from_scene(sc, flags=flags, device=dev, reach_levels=n_cycles if reach else 0)
        self.hard_d = torch.from_numpy(sc.hard).to(dev)
        self.soft_d = torch.from_numpy(sc.soft).to(dev) if sc.soft is not None else None
        self.hard_h = torch.from_numpy(sc.hard).pin_memory()
        self.soft_h = torch.from_numpy(sc.soft).pin_memory() if sc.soft is not None else None
        self.goal, self.plan = tuple(sc.goal), None
        self.n_r = sc.n * sc.n * sc.nt
        self.updates_per_plan = 6 * n_cycles * self.n_r
        I = self.p.debug_tables()["I"]
        self.nx = int((I == 0).sum())                                   # slices swept by the x-rows kernel (eq (19))

    def step(self, hard, soft):
        p, sc, nhp = self.p, self.sc, self.nhp
        if self.reach:
            p.render_obstacles(hard, None if not p.flags & 2 else soft)
            p.reach_run(sc.start, self.n_cycles)
            try:
                self.plan = p.reach_extract_path(self.goal)
            except nhp.NhpError as e:
                if e.code != -5:
                    raise
                self.plan = ([], 0xFFFFFFFF)
            return
        if self.dt_dev:
            p.render_obstacles_dt(hard, 4.0)                       # pipeline steps 1-4 on the device
        else:
            p.render_obstacles(hard, soft)
        p.run_nturn(sc.start, self.n_cycles)
        try:
            self.plan = p.extract_path(self.goal)                  # synchronises; plan comes back to the host
        except nhp.NhpError as e:
            if e.code != -5:
                raise
            self.plan = ([], 0xFFFFFFFF)

    def warm_up(self, n):
        """Warm-up steps, then choose a goal the sweeps actually reach (fixed for all timed steps)."""
        p, sc = self.p, self.sc
        for _ in range(max(n, 1)):
            self.step(self.hard_d, self.soft_d)
        if self.reach:
            K = p.reach_count_numpy()
            cands = [tuple(sc.goal)] + [tuple(g) for g in sc.extra_goals]
            reached = [g for g in cands if K[g[2], g[1], g[0]] != 255]
            self.goal = reached[0] if K[sc.goal[2], sc.goal[1], sc.goal[0]] != 255 or not reached else max(reached, key=lambda g: K[g[2], g[1], g[0]])
        else:
            p.status()
            self.goal = pick_goal(p, sc, self.torch)
        self.step(self.hard_d, self.soft_d)

    def timed(self, steps, host=False, profile=False):
        """-> (device ms over `steps` steps, launches, {slot: (ms, launches)} if profile).  With `profile` every launch is
        bracketed by an event pair and the pool is drained after EVERY step, so no launch goes untimed."""
        p, torch = self.p, self.torch
        hard, soft = (self.hard_h, self.soft_h) if host else (self.hard_d, self.soft_d)
        p.kernel_times(reset=True)
        p.set_profiling(profile)
        l0 = p.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.replicas.barrier(); torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            self.step(hard, soft)
            if profile:
                p.kernel_times()
        e1.record()
        torch.cuda.synchronize(); self.replicas.barrier()
        p.set_profiling(False)
        kt = p.kernel_times(reset=True) if profile else None
        return e0.elapsed_time(e1), p.launch_count() - l0, kt

    def launch_path(self):
        """Which launch sequence the timed pass and the event-bracketed (profiled) pass run (they differ on small grids)."""
        if self.reach:
            return {"timed": "separate launches", "profiled": "separate launches"}
        fl, nhp = self.p.flags, self.nhp
        sparse = not fl & (nhp.FLAG_FIXED_WORK | nhp.FLAG_NO_SHORTCUTS | nhp.FLAG_SIMPLE_KERNELS | nhp.FLAG_FORWARD_ONLY)
        first = "one-tile first LF" if sparse else "full first LF"
        sep = f"separate launches, {first}, " + ("one-band first SF" if sparse else "full first SF")
        g = self.p.cycle_graph_kernels()
        return {"timed": f"CUDA graph of the inner cycle ({g} kernels per replay), {first}, full first SF" if g else sep, "profiled": sep}

    def updates_per_launch(self, slot):
        """Pose-updates one launch of `slot` processes (N_R per maneuver kernel)."""
        nt = self.sc.nt
        return {"turn_pair": 2 * self.n_r, "straight_xrows": self.n_r * self.nx // nt,
                "straight_rows": self.n_r * (nt - self.nx) // nt}.get(slot, self.n_r)

    def rooflines(self, kt, steps, step_ms, peak, config):
        """Per sweep kernel: algorithmic bytes / CUDA-event time (`frac_nominal`, the 6-pass definition of SURVEY 8(d): NOT a
        physical fraction while the short cuts are on) and the committed ncu dram bytes / the same time (`frac_traffic`, the
        physical HBM fraction)."""
        alg_b = ALG_BYTES_SOFT if self.sc.soft is not None else ALG_BYTES_HARD
        out = {}
        for k in SWEEP_SLOTS:
            ms, n = kt.get(k, (0.0, 0))
            if not n:
                continue
            if k == "LF" and not (self.p.flags & (self.nhp.FLAG_FIXED_WORK | self.nhp.FLAG_NO_SHORTCUTS)):
                continue            # the first LF of a plan is one tile (the curve through the start), not a sweep of the volume
            avg = ms / n
            alg = alg_b * self.updates_per_launch(k)
            tr = measured_traffic(config, k)
            ach = alg / (avg * 1e-3) / 1e9
            fresh = tr is not None and not tr["stale"]
            out[k] = {"avg_launch_ms": avg, "launches_timed": int(n), "ms_per_step": ms / steps, "share_of_step": ms / steps / step_ms,
                      "pose_updates_per_launch": self.updates_per_launch(k), "algorithmic_bytes_per_launch": alg,
                      "achieved_nominal": ach, "frac_nominal": ach / peak,
                      "traffic": tr["bytes_per_launch"] if tr else None, "traffic_source": tr["source"] if tr else None,
                      "traffic_stale": tr["stale"] if tr else None,
                      "frac_traffic": (tr["bytes_per_launch"] / (avg * 1e-3) / 1e9 / peak) if fresh else None}
        return out

    def close(self):
        self.p.close()
        del self.hard_d, self.soft_d, self.p
        self.torch.cuda.empty_cache()


def side_config(nhp, torch, replicas, dev, config, peak, flags=0, steps=2, cycles=0, traffic_key=None):
    """One more workload (or the same one under NHP_FLAG_FIXED_WORK), timed the same way with fewer steps."""
    import scenes
    sc = scenes.CONFIGS[config](replicas.replica_seed(config, 0))
    b = PlanBench(nhp, torch, replicas, sc, cycles or sc.n_cycles, dev, flags=flags)
    b.warm_up(1)
    ms, launches, _ = b.timed(steps)
    ms_prof, _, kt = b.timed(steps, profile=True)
    rl = b.rooflines(kt, steps, ms_prof / steps, peak, traffic_key or config)
    dom = max(rl, key=lambda k: rl[k]["ms_per_step"]) if rl else None
    out = {"workload": workload_name(sc, b.n_cycles), "baseline_config": config, "steps": steps, "ms_per_step": ms / steps,
           "value": steps * b.updates_per_plan / (ms * 1e-3) / 1e9, "unit": UNIT, "plans_per_sec": steps / (ms * 1e-3),
           "gpu_launches": int(launches), "plan_waypoints": len(b.plan[0]), "plan_cost": b.plan[1],
           "dominant_kernel": dom,
           "launch_path": b.launch_path(),
           "kernels": {k: {kk: v[kk] for kk in ("avg_launch_ms", "ms_per_step", "frac_nominal", "traffic", "traffic_stale", "frac_traffic")} for k, v in rl.items()},
           "kernel_ms_per_step": {k: round(v[0] / steps, 4) for k, v in kt.items() if v[1] and k not in nhp.binding.NESTED_SLOTS}}
    b.close()
    return out


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` (N > 1) outside torchrun: launch the N ranks ourselves, one process per GPU."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    sys.exit(subprocess.call(cmd))


def run_ours(args):
    if args.gpus > 1 and "RANK" not in os.environ:
        respawn_under_torchrun(args)
    import torch

    import paper_2306_01301_b200 as nhp
    import scenes
    from paper_2306_01301_b200 import replicas

    rank, local_rank, ws = replicas.init("nccl")
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    assert ws == args.gpus, f"--gpus {args.gpus} but WORLD_SIZE = {ws}"
    assert local_rank < torch.cuda.device_count(), f"rank {rank}: only {torch.cuda.device_count()} GPU(s) visible"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    sc = scenes.CONFIGS[args.config](replicas.replica_seed(args.config, rank))
    n_cycles = args.cycles or sc.n_cycles
    flags = (nhp.FLAG_SIMPLE_KERNELS if args.simple_kernels else 0) | (nhp.FLAG_FIXED_WORK if args.fixed_work else 0) | (nhp.FLAG_NO_SHORTCUTS if args.no_shortcuts else 0) | (nhp.FLAG_SECTIONS if args.sections else 0) | (nhp.FLAG_NO_SECTIONS if args.no_sections else 0)
    b = PlanBench(nhp, torch, replicas, sc, n_cycles, dev, flags=flags, reach=args.reach, dt_on_device=args.dt_on_device)
    p, n_r, updates_per_plan, dt_dev = b.p, b.n_r, b.updates_per_plan, b.dt_dev
    b.warm_up(args.warmup)

    clocks = ClockSampler(local_rank)
    if rank == 0:
        clocks.start()
    ms_dev, launches, _ = b.timed(args.steps)
    # the same K steps once more with an event pair around every launch: per-kernel durations for the roofline lines
    # (the events cost ~3 % of the step, so `value` is taken from the pass without them)
    ms_prof, _, kt = b.timed(args.steps, profile=True)
    dropped = p.prof_dropped()
    clk = clocks.stop() if rank == 0 else None
    ms_e2e, _, _ = b.timed(args.steps, host=True)
    plan, cost = b.plan
    ms_dev_max, units = replicas.aggregate(ms_dev, args.steps * updates_per_plan, dev)
    ms_e2e_max, _ = replicas.aggregate(ms_e2e, 0, dev)
    if rank != 0:
        b.close(); replicas.shutdown()
        return

    peak, peak_src = peak_hbm()
    state = {"goal": b.goal, "plan": b.plan}
    hard_h, soft_h = b.hard_h, b.soft_h
    if args.reach:
        return finish_reach(args, sc, n_cycles, n_r, ws, ms_dev_max, ms_e2e_max, units, launches, kt, clk, state, peak, peak_src, hard_h, p, replicas)
    step_prof_ms = ms_prof / args.steps
    if not any(kt.get(k, (0, 0))[1] for k in SWEEP_SLOTS):               # bring-up kernels: the maneuver slots themselves
        rl = {}
        sweeps = {k: v for k, v in kt.items() if k in nhp.MANEUVER_NAMES and v[1]}
    else:
        rl = b.rooflines(kt, args.steps, step_prof_ms, peak, args.config)
        sweeps = {k: kt[k] for k in rl}
    alg_b = ALG_BYTES_SOFT if sc.soft is not None else ALG_BYTES_HARD
    dom = max(sweeps, key=lambda k: sweeps[k][0])
    dom_ms, dom_n = sweeps[dom]
    dom_upd = b.updates_per_launch(dom)
    per_launch_bytes = alg_b * dom_upd
    achieved = per_launch_bytes / (dom_ms / max(dom_n, 1) * 1e-3) / 1e9 if dom_ms > 0 else 0.0
    sweep_ms = sum(v[0] for v in sweeps.values())
    sweep_gbs = alg_b * n_r * 6 * n_cycles * args.steps / (sweep_ms * 1e-3) / 1e9 if sweep_ms > 0 else 0.0
    dom_rl = rl.get(dom, {})
    # physical HBM fraction of all sweeps together: committed ncu dram bytes per launch x launches / their summed time
    tr_known = [k for k in rl if rl[k]["frac_traffic"] is not None]          # captured, and the kernel's source unchanged since
    tr_bytes = sum(rl[k]["traffic"] * rl[k]["launches_timed"] for k in tr_known)
    tr_ms = sum(sweeps[k][0] for k in tr_known)
    # secondary bound: the integer min/max pipe, measured live by the library's micro-benchmark
    sm_clock = (clk or {}).get("sm_mhz") or 1965.0
    alu_ops, sm_count = p.microbench_alu(8)
    alu_peak = alu_ops / 1e12                                                   # T lane-ops / s
    ops_per_update = 3 if dom.startswith("straight") or dom in ("SF", "SB") else 5
    alu_achieved = ops_per_update * dom_upd / (dom_ms / max(dom_n, 1) * 1e-3) / 1e12 if dom_ms > 0 else 0.0
    top_level = {k: v for k, v in kt.items() if v[1] and k not in nhp.binding.NESTED_SLOTS}
    out = {
        "metric": METRIC, "value": units / (ms_dev_max * 1e-3) / 1e9, "unit": UNIT, "n_gpus": ws,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_dev_max / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "value_definition": ("NOMINAL pose-updates (6 * N_T * N_R per plan, PAPER.md:453) / time" +
                             ("; every data-dependent short cut is off in this run" if (args.fixed_work or args.no_shortcuts or args.simple_kernels) else
                              ", data-dependent short cuts ON: tiles without a finite value or fully blocked are skipped, a vertex is stored only "
                              "where it improved, the first LF / SF of a plan touch one tile / one band per slice -- the time depends on the "
                              "scene; the scene-independent figures are fixed_work_* (same instructions and bytes whatever the scene holds, "
                              "PAPER.md:565) and no_shortcuts_*")),
        "launch_path": b.launch_path(),
        "config": bench_config(sc, n_cycles, args, ws, dt_dev),
        "result": {"goal": list(b.goal), "plan_waypoints": len(plan), "plan_cost": cost},
        "plans_per_sec": ws * args.steps / (ms_dev_max * 1e-3),
        "clocks": clk,
        "e2e": {"value": units / (ms_e2e_max * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": ms_e2e_max / args.steps,
                "h2d_bytes_per_step": int(hard_h.numel() + (soft_h.numel() if (soft_h is not None and not dt_dev) else 0)),
                "d2h_bytes_per_step": int(4 * 16 + 16 * max(len(plan), nhp.binding.PLAN_EAGER))},      # status words + the waypoints that travel with them
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "kernel": dom, "pose_updates_per_launch": dom_upd, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": dom_rl.get("traffic"), "frac_traffic": dom_rl.get("frac_traffic"),
                     "traffic_source": dom_rl.get("traffic_source"), "peak_source": peak_src,
                     "frac_definition": "frac = SURVEY 8(d) algorithmic bytes (8.125 B, 9.125 B soft, per NOMINAL pose-update; a fused pair launch is "
                                        "charged two maneuvers) / CUDA-event time / peak.  It is the contract's 6-pass figure, not a physical fraction: it "
                                        "exceeds 1 because the kernels move fewer bytes than the definition charges -- in every kernel the 4-byte write "
                                        "happens only where a vertex improved and tiles with nothing to do are skipped (this alone puts the straight "
                                        "kernels, which fuse nothing, above 1), the collision bit is stamped into V (no separate read), and a turn-pair "
                                        "launch reads V once for the four laps of two maneuvers.  frac_traffic = ncu dram bytes per launch "
                                        "(profiles/traffic.csv, captured at traffic_commit; null when the kernel's source changed since) / the same "
                                        "time / peak: the physical HBM fraction.  Per-kernel rows carry the 6-pass figure as frac_nominal.",
                     "traffic_commit": traffic_table()[2], "traffic_stale": dom_rl.get("traffic_stale"),
                     "algorithmic_bytes_per_launch": per_launch_bytes, "avg_launch_ms": dom_ms / max(dom_n, 1),
                     "launches_timed": int(dom_n), "launches_untimed": int(dropped),
                     "kernels": rl,
                     "all_sweeps": {"achieved": sweep_gbs, "frac": sweep_gbs / peak, "ms_per_step": sweep_ms / args.steps,
                                    "traffic_per_step": tr_bytes / args.steps if tr_known else None,
                                    "frac_traffic": (tr_bytes / (tr_ms * 1e-3) / 1e9 / peak) if tr_known and tr_ms > 0 else None}},
        "alu": {"bound": "alu", "kernel": dom, "achieved": alu_achieved, "peak": alu_peak, "unit": "T min/max lane-ops/s",
                "frac": alu_achieved / alu_peak, "ops_per_pose_update": ops_per_update,
                "peak_source": f"nhp_microbench_alu, measured in this run: 8 independent VIADDMNMX chains per thread, 8 warps per sub-partition, "
                               f"{sm_count} SMs = {alu_ops / (sm_count * 4 * sm_clock * 1e6):.2f} lane-ops per sub-partition and clock at {sm_clock:.0f} MHz (DESIGN.md 6.7)"},
        "read_probe_gbs": {name: (p.microbench_read(k) / 1e9 if k < 3 or p.nt <= 1024 else None)       # the turn-tile pattern is one CTA of N_theta threads
                           for k, name in enumerate(("linear", "rows_pattern", "xrows_pattern", "turn_tile_pattern"))},
        "kernel_ms_per_step": {k: round(v[0] / args.steps, 4) for k, v in top_level.items()},
        "kernel_ms_sum": sum(v[0] for v in top_level.values()) / args.steps,
        "ms_per_step_with_kernel_events": step_prof_ms,
    }
    b.close()
    rf = out["roofline"]
    rf["frac_traffic_all_sweeps"] = rf["all_sweeps"]["frac_traffic"]          # scalar copies: the driver's record keeps scalars only
    rf["traffic_per_step"] = rf["all_sweeps"]["traffic_per_step"]
    if ws == 1 and not args.no_extra:
        # T12 ("run time independent of scene"): the same workload with the data-dependent short cuts off
        if not args.fixed_work and not args.no_shortcuts and not args.simple_kernels:
            for key, fl, cfgkey in (("no_shortcuts", nhp.FLAG_NO_SHORTCUTS, f"{args.config}:no_shortcuts"), ("fixed_work", nhp.FLAG_FIXED_WORK, f"{args.config}:fixed_work")):
                fw = side_config(nhp, torch, replicas, dev, args.config, peak, flags=fl, steps=min(args.steps, 3), cycles=args.cycles, traffic_key=cfgkey)
                out[key] = {k: fw[k] for k in ("ms_per_step", "value", "unit", "plans_per_sec", "steps", "kernels")}
                out[f"{key}_ms_per_step"] = rf[f"{key}_ms_per_step"] = fw["ms_per_step"]
                out[f"{key}_value"] = fw["value"]
                # whole plan against the 6-pass definition: with NHP_FLAG_FIXED_WORK the definition's bytes are (at least) moved
                rf[f"{key}_frac"] = alg_b * 6 * n_cycles * n_r / (fw["ms_per_step"] * 1e-3) / 1e9 / peak
                kn = fw["kernels"]
                known = [k for k in kn if kn[k]["frac_traffic"] is not None]
                t_ms = sum(kn[k]["ms_per_step"] for k in known)
                rf[f"{key}_frac_traffic_all_sweeps"] = (sum(kn[k]["frac_traffic"] * kn[k]["ms_per_step"] for k in known) / t_ms) if known else None
            out["no_shortcuts"]["what"] = "NHP_FLAG_NO_SHORTCUTS: every warp runs every pass of every sweep; vertices written only where they improved"
            out["fixed_work"]["what"] = "NHP_FLAG_FIXED_WORK: no short cuts and every visited vertex written back (the paper's unconditional store): same instructions and bytes whatever the scene holds"
        # the other configurations of BASELINE.json (small grids, the soft-cost path, the largest grid), one short timed run each
        out["other_configs"] = [side_config(nhp, torch, replicas, dev, c, peak, steps=2 if c > 2 else 20) for c in (1, 2, 4, 5) if c != args.config]
        for oc in out["other_configs"]:
            rf[f"cfg{oc['baseline_config']}_ms_per_step"] = oc["ms_per_step"]
            dk = oc["kernels"].get(oc["dominant_kernel"] or "", {})
            rf[f"cfg{oc['baseline_config']}_frac_traffic"] = dk.get("frac_traffic")
        # the reachability planner of appendix C on the same workload (Table 9)
        rb = PlanBench(nhp, torch, replicas, scenes.CONFIGS[args.config](replicas.replica_seed(args.config, 0)), n_cycles, dev, reach=True)
        rb.warm_up(1)
        r_ms, r_launches, _ = rb.timed(3)
        out["reach"] = {"what": f"reachability (bit-vector) planner, appendix C: render + {n_cycles} levels + back-track on config {args.config}",
                        "ms_per_step": r_ms / 3, "steps": 3, "gpu_launches": int(r_launches), "plan_waypoints": len(rb.plan[0]), "plan_maneuvers": rb.plan[1]}
        rf["reach_ms_per_step"] = out["reach_ms_per_step"] = r_ms / 3
        rb.close()
    if not args.no_cpu_baseline and ws == 1:
        out["cpu_baseline"] = cpu_baseline(sc, n_cycles, sample_cycles=2)
    replicas.shutdown()
    print(json.dumps(out), flush=True)


def finish_reach(args, sc, n_cycles, n_r, ws, ms_dev_max, ms_e2e_max, units, launches, kt, clk, state, peak, peak_src, hard_h, p, replicas):
    """JSON line of the reachability planner (appendix C): same metric, a pose-update = one bit visited by one maneuver sweep
    of one level; algorithmic bytes per pose-update = read the level bit + the collision bit, write the next level's bit."""
    lv_ms, lv_n = kt.get("reach_level", (0.0, 0))
    per_launch_bytes = 0.375 * 6 * n_r
    achieved = per_launch_bytes / (lv_ms / max(lv_n, 1) * 1e-3) / 1e9 if lv_ms > 0 else 0.0
    plan, nm = state["plan"]
    out = {
        "metric": METRIC.replace("N-turn planner", "reachability (bit-vector) planner, appendix C"), "value": units / (ms_dev_max * 1e-3) / 1e9,
        "unit": UNIT, "n_gpus": ws, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_dev_max / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u1 (bit per pose)", "data": "synthetic",
        "config": {"workload": workload_name(sc, n_cycles) + ", reachability planner: N_T levels", "baseline_config": args.config,
                   "goal": list(state["goal"]), "plan_waypoints": len(plan), "plan_maneuvers": nm,
                   "l2": "level volumes of %.0f MiB each: L2-resident; HBM roofline shown for orientation only" % (n_r / 8 / 2**20)},
        "plans_per_sec": ws * args.steps / (ms_dev_max * 1e-3), "clocks": clk,
        "e2e": {"value": units / (ms_e2e_max * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": ms_e2e_max / args.steps,
                "h2d_bytes_per_step": int(hard_h.numel()), "d2h_bytes_per_step": int(16 * 4096 + 32)},
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "kernel": "reach_level (one level: six maneuver sweeps, copies, transpositions)", "achieved": achieved,
                     "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": per_launch_bytes, "avg_launch_ms": lv_ms / max(lv_n, 1), "launches_timed": int(lv_n)},
        "kernel_ms_per_step": {k: round(v[0] / args.steps, 4) for k, v in kt.items() if v[1]},
    }
    p.close()
    replicas.shutdown()
    print(json.dumps(out), flush=True)


def oracle_setup(sc):
    """Oracle handle plus its own rendering of the scene (the oracle never sees anything from the CUDA path)."""
    import oracle
    o = oracle.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct, sc.dir_mult, sc.cost_one_log2, sc.flags, threads=0)
    fp = oracle.Footprint(sc.mask, sc.ou, sc.ov)
    t0 = time.perf_counter()
    Cv, Sv = o.render(fp, sc.hard, sc.soft, method="runs")
    return o, Cv, Sv, time.perf_counter() - t0


def cpu_baseline(sc, n_cycles, sample_cycles=2):
    """The oracle as it stands on this box's host cores, on a bounded sample of the same workload: its own
    rendering of the scene plus `sample_cycles` of the N_T maneuver cycles over the full volume.  The value is
    plan-equivalent: sampled pose-updates / (sweep time + render time * sample_cycles / N_T).  `single_thread` is the
    same oracle on ONE thread (the configuration of the paper's CPU rows) over two maneuver sweeps."""
    import numpy as np
    o, Cv, Sv, t_render = oracle_setup(sc)
    V = np.full(o.shape, 0xFFFFFFFF, np.uint32)
    V[sc.start[2], sc.start[1], sc.start[0]] = 0
    t0 = time.perf_counter()
    o.cycles(V, Cv, Sv, sample_cycles)
    t_sweeps = time.perf_counter() - t0
    upd = 6 * sample_cycles * V.size
    cores = int(o.threads)
    o.set_threads(1)
    t0 = time.perf_counter()
    o.sweep(0, V, Cv, Sv)                              # LF: a turn maneuver (two laps)
    o.sweep(1, V, Cv, Sv)                              # SF: a straight maneuver
    t_one = time.perf_counter() - t0
    return {"value": upd / (t_sweeps + t_render * sample_cycles / n_cycles) / 1e9, "unit": UNIT, "cores": cores,
            "kind": "oracle",
            "sample": f"oracle render of the full scene ({t_render:.2f} s) + {sample_cycles} of {n_cycles} maneuver cycles "
                      f"over the full {sc.n}x{sc.n}x{sc.nt} volume ({t_sweeps:.2f} s), OpenMP over curves on all host cores; "
                      f"render time charged pro rata",
            "single_thread": {"value": 2 * V.size / t_one / 1e9, "unit": UNIT, "cores": 1,
                              "sample": f"one turn sweep (LF) + one straight sweep (SF) over the full volume on one thread ({t_one:.2f} s), "
                                        f"sweeps only (no render)"}}


def run_reference(args):
    """--impl reference: the CPU oracle (the only 'reference' this tier has), one bounded sample per step."""
    from paper_2306_01301_b200 import replicas
    rank, _, ws = replicas.world()
    if rank != 0:
        return
    import numpy as np

    import scenes
    sc = scenes.get_config(args.config)
    n_cycles = args.cycles or sc.n_cycles
    o, Cv, Sv, t_render = oracle_setup(sc)
    V = np.full(o.shape, 0xFFFFFFFF, np.uint32)
    V[sc.start[2], sc.start[1], sc.start[0]] = 0
    whole_cycle = (args.steps + args.warmup) <= 12
    fwd_only = bool(sc.flags & 1)

    def step(k):
        if whole_cycle:
            o.cycles(V, Cv, Sv, 1)
            return (3 if fwd_only else 6) * V.size
        o.sweep(k % 6, V, Cv, Sv)
        return V.size

    for k in range(args.warmup):
        step(k)
    t0 = time.perf_counter()
    upd = sum(step(args.warmup + k) for k in range(args.steps))
    dt = time.perf_counter() - t0
    val = upd / dt / 1e9
    sample = (("one maneuver cycle (6 sweeps)" if whole_cycle else "one maneuver sweep (maneuver = step mod 6)") +
              f" over the full {sc.n}x{sc.n}x{sc.nt} volume per step; scene rendered once by the oracle before timing "
              f"({t_render:.2f} s, not in the value)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": ws, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": bench_config(sc, n_cycles, args, ws),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": int(o.threads), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
