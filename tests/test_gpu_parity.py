"""GPU <-> oracle parity through the C ABI (bit-exact: costs are integers, plans identical)."""
import numpy as np
import pytest

import scenes

pytestmark = pytest.mark.gpu

INF = 0xFFFFFFFF


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import oracle
    import paper_2306_01301_b200 as nhp
    oracle.build()
    nhp.load_library()
    return oracle, nhp


def oracle_for(oracle, sc, threads=0):
    o = oracle.Oracle(sc.log2_n, sc.log2_nt, sc.R, sc.ct, sc.dir_mult, sc.cost_one_log2, sc.flags, threads=threads)
    return o, oracle.Footprint(sc.mask, sc.ou, sc.ov)


def small_scenes():
    return [
        scenes.random_scene(5, 5, 4, 1),
        scenes.random_scene(5, 5, 4, 2, soft=True, reverse_mult=512),
        scenes.random_scene(5, 6, 7.3, 3, vehicle=(6, 3), soft=True),
        scenes.random_scene(6, 5, 5, 4, vehicle=(7, 3), n_rects=12),
        scenes.random_scene(6, 6, 8, 5, flags=1, soft=True),                       # forward only
        scenes.random_scene(5, 7, 4, 6, ct=(4096, 0, 5000, 5000, 0, 4096)),        # N_theta > N, compact weights
        scenes.random_scene(7, 6, 9, 7, vehicle=(9, 4), n_rects=20, soft=True, reverse_mult=300, n_cycles=2),
        scenes.random_scene(5, 10, 6, 8, n_cycles=2),                                # N_theta = 1024: 32 sections, 1024-thread tiles
        scenes.random_scene(5, 10, 5, 9, soft=True, reverse_mult=400, n_cycles=2),
        scenes.random_scene(8, 5, 4.5, 10, vehicle=(3, 2), n_rects=40, n_cycles=2),  # N = 256, N_theta = 32: one section per curve
    ]


@pytest.mark.parametrize("flags", [0, 4, 8, 16, 64, 64 | 8])     # tile kernels (straight sweeps by Sections at these sizes), thread-per-curve kernels,
                                                                  # NHP_FLAG_FIXED_WORK, NHP_FLAG_NO_SHORTCUTS, NHP_FLAG_NO_SECTIONS (streaming straight kernels), the same with fixed work
def test_tables_render_sweeps_and_plans_match_the_oracle(mods, flags):
    oracle, nhp = mods
    for sc in small_scenes():
        o, fp = oracle_for(oracle, sc)
        p = nhp.Planner.from_scene(sc, flags=flags)
        # tables
        t = p.debug_tables()
        for k in ("beta", "psi2", "B", "I", "J", "len_q"):
            assert (t[k] == getattr(o, k)).all(), (sc.name, k)
        # rendering (a1, a2): brute-force oracle
        Cv, Sv = o.render(fp, sc.hard, sc.soft, method="brute")
        p.render_obstacles(sc.hard, sc.soft)
        assert (p.collision_numpy() == Cv).all(), sc.name
        if sc.soft is not None:
            assert (p.soft_numpy() == Sv).all(), sc.name
        # sweeps (a3-a6), one cycle at a time
        p.run_nturn(sc.start, 1)
        V = o.run(Cv, Sv, sc.start, 1)
        assert (p.cost_volume_numpy() == V).all(), sc.name
        for _ in range(sc.n_cycles):
            p.run_more(1)
            o.cycles(V, Cv, Sv, 1)
            got = p.cost_volume_numpy()
            assert (got == V).all(), (sc.name, int((got != V).sum()))
        p.run_nturn(sc.start, sc.n_cycles + 1)
        assert (p.cost_volume_numpy() == V).all(), sc.name
        # back-tracking (a7): identical plans on sampled goals, before and after cost_volume conversion
        rng = np.random.default_rng(1)
        tj, jj, ij = np.nonzero(Cv == 0)
        for k in rng.integers(len(tj), size=40):
            goal = (int(ij[k]), int(jj[k]), int(tj[k]))
            try:
                want = o.backtrack(V, Cv, Sv, sc.start, goal)
            except oracle.OracleError as e:
                with pytest.raises(nhp.NhpError) as g:
                    p.extract_path(goal)
                assert g.value.code == e.code == -5
                continue
            assert p.extract_path(goal) == want, (sc.name, goal)
        p.close()


def test_single_maneuver_sweeps_on_random_volumes(mods):
    """Each maneuver kernel alone, on a volume with arbitrary values (not produced by a run)."""
    oracle, nhp = mods
    # exercised through run_more after uploading a random canonical volume into V
    import torch
    sc = scenes.random_scene(6, 6, 8, 11, soft=True, reverse_mult=512, vehicle=(5, 2), n_rects=10)
    o, fp = oracle_for(oracle, sc)
    Cv, Sv = o.render(fp, sc.hard, sc.soft)
    p = nhp.Planner.from_scene(sc)
    p.render_obstacles(sc.hard, sc.soft)
    p.run_nturn(sc.start, 1)
    rng = np.random.default_rng(2)
    for trial, vmax in enumerate((50000, 1 << 29, (1 << 30) - 1)):
        V = rng.integers(0, vmax, size=o.shape).astype(np.uint32)
        V[rng.random(o.shape) < 0.4] = INF
        V[Cv != 0] = INF
        p.cost_volume().copy_(torch.from_numpy(V.view(np.int32)).to(p.device))
        p.run_more(1)
        o.cycles(V, Cv, Sv, 1)
        assert (p.cost_volume_numpy() == V).all(), trial
    p.close()


def test_distance_transform_and_soft_image_on_the_device(mods):
    """Steps 1-2 of PAPER.md:388-389 on the GPU (nhp_render_obstacles_dt) against the oracle: squared distances are
    integers (the float32 distance is exact-to-rounding, tolerance 1e-5 as north_star asks), the soft image and
    everything rendered and swept from it are bit-exact (rint is taken in float32 on both sides)."""
    oracle, nhp = mods
    import torch
    cases = [scenes.random_scene(5, 5, 4, 21, soft=True), scenes.random_scene(7, 6, 9, 22, vehicle=(6, 3), n_rects=25, soft=True),
             scenes.random_scene(6, 6, 8, 23, n_rects=0, soft=True), scenes.get_config(4)]
    for sc in cases:
        for k in (4.0, 0.0, 11.5):
            d2, dist, soft = oracle.soft_from_hard(sc.hard, k)
            p = nhp.Planner.from_scene(sc)
            dist_g = torch.empty((sc.n, sc.n), dtype=torch.float32, device=p.device)
            p.render_obstacles_dt(sc.hard, k, dist_g)
            got = dist_g.cpu().numpy()
            assert np.allclose(got, dist, rtol=1e-5, atol=1e-5), sc.name
            assert (got == dist).all(), sc.name                      # in fact bit-equal: sqrt of the same integer, rounded once
            assert (p.soft_image_numpy() == soft).all(), (sc.name, k)
            if sc.n <= 128 and k == 4.0:
                o, fp = oracle_for(oracle, sc)
                Cv, Sv = o.render(fp, sc.hard, soft, method="brute")
                assert (p.collision_numpy() == Cv).all() and (p.soft_numpy() == Sv).all(), sc.name
                p.run_nturn(sc.start, 2)
                assert (p.cost_volume_numpy() == o.run(Cv, Sv, sc.start, 2)).all(), sc.name
            if sc.n > 128 and k == 4.0:
                # two cycles swept from the device-made soft image at full size (config 4)
                o, fp = oracle_for(oracle, sc)
                Cv, Sv = o.render(fp, sc.hard, soft, method="runs")
                assert (p.collision_numpy() == Cv).all() and (p.soft_numpy() == Sv).all(), sc.name
                p.run_nturn(sc.start, 2)
                assert (p.cost_volume_numpy() == o.run(Cv, Sv, sc.start, 2)).all(), sc.name
            p.close()
            if sc.n > 128:
                break
    # a planner without a soft volume refuses
    sc = scenes.random_scene(5, 5, 4, 1)
    p = nhp.Planner.from_scene(sc)
    with pytest.raises(nhp.NhpError) as e:
        p.render_obstacles_dt(sc.hard, 4.0)
    assert e.value.code == -1
    p.close()


def test_reachability_planner_of_appendix_c(mods):
    """Bit-vector planner: fewest-maneuver counts from the level volumes and the plans extracted over
    them against the oracle, bit for bit, incl. forward-only, N_theta != N and config 2."""
    oracle, nhp = mods
    rng = np.random.default_rng(13)
    cases = [(scenes.random_scene(5, 5, 4, 61, n_rects=5), 12), (scenes.random_scene(6, 5, 5, 62, vehicle=(6, 3), n_rects=12), 6),
             (scenes.random_scene(5, 7, 4, 63), 5), (scenes.random_scene(6, 6, 8, 64, flags=1), 7), (scenes.random_scene(7, 6, 9, 65, n_rects=30), 4),
             (scenes.get_config(2), 6)]
    for sc, n_levels in cases:
        o, fp = oracle_for(oracle, sc)
        Cv, _ = o.render(fp, sc.hard, None, method="runs")
        K = o.reach_run(Cv, sc.start, n_levels)
        p = (nhp.Planner.from_scene(sc, reach_levels=n_levels) if sc.soft is None else
             nhp.Planner(sc.log2_n, sc.log2_nt, sc.R, sc.ct, flags=sc.flags & 1, reach_levels=n_levels))
        if sc.soft is not None:
            p.render_vehicle_footprint(sc.mask, sc.ou, sc.ov)
        p.render_obstacles(sc.hard)
        p.reach_run(sc.start, n_levels)
        got = p.reach_count_numpy()
        assert (got == K).all(), (sc.name, int((got != K).sum()))
        tj, jj, ij = np.nonzero(K != 255)
        for k in rng.integers(len(tj), size=30):
            goal = (int(ij[k]), int(jj[k]), int(tj[k]))
            assert p.reach_extract_path(goal) == o.reach_backtrack(K, Cv, sc.start, goal), (sc.name, goal)
        tj, jj, ij = np.nonzero((K == 255) & (Cv == 0))
        if len(tj):
            with pytest.raises(nhp.NhpError) as e:
                p.reach_extract_path((int(ij[0]), int(jj[0]), int(tj[0])))
            assert e.value.code == -5
        # a second, shorter run reuses the buffers; more levels than the planner was created for are refused
        p.reach_run(sc.start, 2)
        assert (p.reach_count_numpy() == o.reach_run(Cv, sc.start, 2)).all()
        with pytest.raises(nhp.NhpError) as e:
            p.reach_run(sc.start, n_levels + 1)
        assert e.value.code == -6
        p.close()


@pytest.mark.slow
def test_reachability_planner_config3_maze_512(mods):
    """Full size, the launch configuration `bench.py --reach` times: 20 levels at 512^3."""
    oracle, nhp = mods
    sc = scenes.get_config(3)
    o, fp = oracle_for(oracle, sc)
    Cv, _ = o.render(fp, sc.hard, None, method="runs")
    K = o.reach_run(Cv, sc.start, sc.n_cycles)
    p = nhp.Planner.from_scene(sc, reach_levels=sc.n_cycles)
    p.render_obstacles(sc.hard)
    p.reach_run(sc.start, sc.n_cycles)
    got = p.reach_count_numpy()
    assert (got == K).all(), int((got != K).sum())
    far = np.argwhere(K == K[K != 255].max())
    for t, j, i in far[:: max(1, len(far) // 8)][:8]:
        goal = (int(i), int(j), int(t))
        assert p.reach_extract_path(goal) == o.reach_backtrack(K, Cv, sc.start, goal), goal
    p.close()


def test_footprint_elements_match_the_oracle(mods):
    """The structuring elements E_Theta (DESIGN R15) through nhp_debug_footprint against the oracle's orc_footprint_offsets,
    at every Theta: box vehicles, a mask with a hole and a notch, a fractional origin."""
    oracle, nhp = mods
    holed = np.ones((5, 9), np.uint8)
    holed[2, 3:6] = 0
    holed[0, 0] = 0
    cases = [(5, 5, 4, np.ones((2, 4), np.uint8), 0.3, 0.5), (6, 6, 8, np.ones((3, 7), np.uint8), 0.9, 1.0), (5, 7, 4, holed, 2.25, 1.75),
             (7, 6, 9, np.ones((9, 20), np.uint8), 3.5, 4.0)]
    for log2_n, log2_nt, R, mask, ou, ov in cases:
        o = oracle.Oracle(log2_n, log2_nt, R, (1024,) * 6)
        fp = oracle.Footprint(mask, ou, ov)
        p = nhp.Planner(log2_n, log2_nt, R, (1024,) * 6)
        p.render_vehicle_footprint(mask, ou, ov)
        rad, cov = p.debug_footprint()
        assert rad == fp.radius()
        for t in range(o.nt):
            da, db = o.footprint_offsets(fp, t)
            want = np.zeros((2 * rad + 1, 2 * rad + 1), np.uint8)
            want[db + rad, da + rad] = 1
            assert (cov[t] == want).all(), (mask.shape, t)
        p.close()
    # a footprint beyond the limit the planner was created for is refused, and so is one that does not fit the grid
    p = nhp.Planner(7, 6, 9, (1024,) * 6, max_footprint_radius=8)
    with pytest.raises(nhp.NhpError) as e:
        p.render_vehicle_footprint(np.ones((9, 20), np.uint8), 3.5, 4.0)
    assert e.value.code == -6
    p.set_box(4, 1, 1)
    p.close()


def test_the_two_planners_keep_their_state_apart(mods):
    """One handle runs the N-turn planner and the reachability planner in any order: a blocked start of one must not leak
    into the other, and a new rendering invalidates the results of both."""
    oracle, nhp = mods
    sc = scenes.random_scene(6, 5, 5, 71, n_rects=8)
    o, fp = oracle_for(oracle, sc)
    Cv, _ = o.render(fp, sc.hard, None, method="brute")
    blocked = (0, 7, 3)                                               # wall cell
    p = nhp.Planner.from_scene(sc, reach_levels=6)
    p.render_obstacles(sc.hard)
    V = o.run(Cv, None, sc.start, 3)
    K = o.reach_run(Cv, sc.start, 6)
    tj, jj, ij = np.nonzero((V != INF) & (K != 255))
    goal = (int(ij[len(ij) // 2]), int(jj[len(ij) // 2]), int(tj[len(ij) // 2]))
    # N-turn run from a good start, then a reachability run from a blocked one
    p.run_nturn(sc.start, 3)
    p.reach_run(blocked, 6)
    with pytest.raises(nhp.NhpError) as e:
        p.reach_extract_path(goal)
    assert e.value.code == -4
    p.status()                                                        # the N-turn run is not affected
    assert p.extract_path(goal) == o.backtrack(V, Cv, None, sc.start, goal)
    # and the other way round
    p.reach_run(sc.start, 6)
    p.run_nturn(blocked, 3)
    with pytest.raises(nhp.NhpError) as e:
        p.extract_path(goal)
    assert e.value.code == -4
    assert p.reach_extract_path(goal) == o.reach_backtrack(K, Cv, sc.start, goal)
    # a new rendering: neither planner may back-track its old volumes against the new collision volume
    p.run_nturn(sc.start, 3)
    p.render_obstacles(np.zeros_like(sc.hard))
    for call in (lambda: p.extract_path(goal), lambda: p.reach_extract_path(goal), lambda: p.reach_count_numpy(), lambda: p.cost_volume()):
        with pytest.raises(nhp.NhpError) as e:
            call()
        assert e.value.code == -8
    p.render_vehicle_footprint(sc.mask, sc.ou, sc.ov)                # a new footprint invalidates the rendering as well
    with pytest.raises(nhp.NhpError) as e:
        p.run_nturn(sc.start, 1)
    assert e.value.code == -8
    p.close()


def test_no_device_allocation_after_create(mods):
    """PAPER.md:565 "no memory allocation takes place during processing": after nhp_planner_create (and one warm-up plan,
    which loads the kernels' code) a footprint change, rendering, both planners and path extraction leave the device's free
    memory where it was."""
    oracle, nhp = mods
    import torch
    sc = scenes.random_scene(7, 6, 9, 72, vehicle=(9, 4), n_rects=20, soft=True, reverse_mult=300, n_cycles=2)
    p = nhp.Planner.from_scene(sc, reach_levels=5)
    K = torch.empty(p.shape, dtype=torch.uint8, device=p.device)

    def everything():
        p.render_vehicle_footprint(sc.mask, sc.ou, sc.ov)
        p.render_obstacles(sc.hard, sc.soft)
        p.render_obstacles_dt(sc.hard, 4.0)
        p.run_nturn(sc.start, 2)
        p.run_nturn_from(sc.start, 1, 1)
        p.run_more(1)
        p.cost_volume()
        p.status()
        try:
            p.extract_path(sc.goal)
            p.extract_path_goalset([sc.goal], 3, 10, 10)
        except nhp.NhpError as e:
            assert e.code == -5
        p.reach_run(sc.start, 5)
        p._check(p._L.nhp_reach_count_volume(p._h, K.data_ptr()), "reach_count_volume")
        try:
            p.reach_extract_path(sc.goal)
        except nhp.NhpError as e:
            assert e.code == -5
        torch.cuda.synchronize()

    everything()
    free0, _ = torch.cuda.mem_get_info()
    everything()
    everything()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    p.close()


def test_default_cycles_and_long_plans(mods):
    """n_cycles <= 0 selects the paper's default of 8 cycles; a plan longer than the waypoints that travel with
    the status words comes back complete (second copy)."""
    oracle, nhp = mods
    sc = scenes.random_scene(6, 6, 8, 73, n_rects=14)
    o, fp = oracle_for(oracle, sc)
    Cv, _ = o.render(fp, sc.hard, None, method="brute")
    V = o.run(Cv, None, sc.start, 8)
    p = nhp.Planner.from_scene(sc)
    p.debug_set_plan_eager(2)
    p.render_obstacles(sc.hard)
    p.run_nturn(sc.start, 0)
    assert (p.cost_volume_numpy() == V).all()
    tj, jj, ij = np.nonzero(V != INF)
    order = np.argsort(V[tj, jj, ij])[::-1][:20]                     # the most expensive goals have the longest plans
    longest = 0
    for k in order:
        goal = (int(ij[k]), int(jj[k]), int(tj[k]))
        want = o.backtrack(V, Cv, None, sc.start, goal)
        assert p.extract_path(goal) == want
        longest = max(longest, len(want[0]))
    assert longest > 3
    p.close()


def test_bounding_box_vehicle_of_appendix_g(mods):
    """nhp_set_box(f, r, s) == the rectangle u in [-r, f), v in [-s, s): collision volume against the
    oracle's brute-force rendering of that rectangle as a mask."""
    oracle, nhp = mods
    sc = scenes.random_scene(6, 6, 8, 51, n_rects=8)
    o, _ = oracle_for(oracle, sc)
    for f, r, s in ((5, 1, 1), (8, 2, 2), (3, 0, 1), (6, 3, 3)):
        fp = oracle.Footprint(np.ones((2 * s, f + r), np.uint8), r - 0.5, s - 0.5)
        Cv, _ = o.render(fp, sc.hard, None, method="brute")
        p = nhp.Planner(sc.log2_n, sc.log2_nt, sc.R, sc.ct)
        p.set_box(f, r, s)
        p.render_obstacles(sc.hard)
        assert (p.collision_numpy() == Cv).all(), (f, r, s)
        p.close()
    with pytest.raises(nhp.NhpError) as e:
        p = nhp.Planner(sc.log2_n, sc.log2_nt, sc.R, sc.ct)
        p.set_box(0, 0, 1)
    assert e.value.code == -1


def test_start_state_with_a_maneuver_in_progress(mods):
    """Section XII: no transition cost for the maneuver in progress at the start; volumes and plans
    against the oracle for every maneuver id."""
    oracle, nhp = mods
    rng = np.random.default_rng(9)
    for sc in (scenes.random_scene(5, 5, 4, 41, n_rects=5, n_cycles=3, soft=True, reverse_mult=384),
               scenes.random_scene(7, 6, 9, 42, vehicle=(6, 3), n_rects=20, n_cycles=2), scenes.random_scene(6, 6, 8, 43, flags=1, n_cycles=2)):
        o, fp = oracle_for(oracle, sc)
        Cv, Sv = o.render(fp, sc.hard, sc.soft, method="runs")
        p = nhp.Planner.from_scene(sc)
        p.render_obstacles(sc.hard, sc.soft)
        for m0 in range(-1, 6):
            if (sc.flags & 1) and m0 in (2, 4, 5):
                with pytest.raises(nhp.NhpError) as e:
                    p.run_nturn_from(sc.start, m0, sc.n_cycles)
                assert e.value.code == -1
                continue
            V = o.run_from(Cv, Sv, sc.start, m0, sc.n_cycles)
            p.run_nturn_from(sc.start, m0, sc.n_cycles)
            got = p.cost_volume_numpy()
            assert (got == V).all(), (sc.name, m0, int((got != V).sum()))
            tj, jj, ij = np.nonzero(V != INF)
            for k in rng.integers(len(tj), size=15):
                goal = (int(ij[k]), int(jj[k]), int(tj[k]))
                assert p.extract_path(goal) == o.backtrack_from(V, Cv, Sv, sc.start, m0, goal), (sc.name, m0, goal)
        p.run_nturn(sc.start, 1)                                  # a plain run afterwards forgets the maneuver
        assert (p.cost_volume_numpy() == o.run(Cv, Sv, sc.start, 1)).all()
        p.close()


def test_goal_search_over_goal_sets(mods):
    """Step 6 (section IX) on the GPU against the oracle: same winner, same score, and the plan
    extracted from it is the oracle's plan from that vertex."""
    oracle, nhp = mods
    rng = np.random.default_rng(7)
    for sc in (scenes.random_scene(6, 5, 5, 31, n_rects=8, n_cycles=4), scenes.random_scene(6, 6, 8, 32, soft=True, reverse_mult=512, n_cycles=3),
               scenes.get_config(2)):
        o, fp = oracle_for(oracle, sc)
        Cv, Sv = o.render(fp, sc.hard, sc.soft, method="runs")
        V = o.run(Cv, Sv, sc.start, sc.n_cycles)
        p = nhp.Planner.from_scene(sc)
        p.render_obstacles(sc.hard, sc.soft)
        p.run_nturn(sc.start, sc.n_cycles)
        tj, jj, ij = np.nonzero(V != INF)
        picks = rng.integers(len(tj), size=24)
        goals = [(int(ij[k]), int(jj[k]), int(tj[k])) for k in picks] + [tuple(sc.goal), (1, 1, 0), (sc.n - 1, sc.n - 2, sc.nt - 1)]
        for trial, g in enumerate(goals):
            d, W, w = int(rng.integers(0, 6)), int(rng.integers(0, 3000)), int(rng.integers(0, 3000))
            gs = [g] if trial % 3 else [g, goals[(trial + 5) % len(goals)], goals[(trial + 11) % len(goals)]]
            try:
                cell, gi, score = o.goal_search(V, gs, d, W, w)
            except oracle.OracleError as e:
                with pytest.raises(nhp.NhpError) as ge:
                    p.extract_path_goalset(gs, d, W, w)
                assert ge.value.code == e.code == -5
                continue
            plan, cost, gcell, ggi, gscore = p.extract_path_goalset(gs, d, W, w)
            assert (gcell, ggi, gscore) == (cell, gi, score), (sc.name, gs, d, W, w)
            assert (plan, cost) == o.backtrack(V, Cv, Sv, sc.start, cell), (sc.name, cell)
        # d = 0, one goal == extract_path
        g = goals[0]
        assert p.extract_path_goalset([g], 0, 5, 5)[:2] == p.extract_path(g)
        with pytest.raises(nhp.NhpError) as ge:
            p.extract_path_goalset([g], 40, 1, 1)
        assert ge.value.code == -1
        p.close()


def test_errors_and_degenerate_cases(mods):
    oracle, nhp = mods
    sc = scenes.random_scene(5, 5, 4, 1)
    p = nhp.Planner(sc.log2_n, sc.log2_nt, sc.R, sc.ct)
    with pytest.raises(nhp.NhpError) as e:
        p.render_obstacles(sc.hard)
    assert e.value.code == -8                                     # no footprint yet
    p.render_vehicle_footprint(sc.mask, sc.ou, sc.ov)
    with pytest.raises(nhp.NhpError) as e:
        p.run_nturn(sc.start, 1)
    assert e.value.code == -8                                     # no render yet
    p.render_obstacles(sc.hard)
    with pytest.raises(nhp.NhpError) as e:
        p.extract_path(sc.goal)
    assert e.value.code == -8
    with pytest.raises(nhp.NhpError) as e:
        p.run_nturn((40, 3, 3), 1)
    assert e.value.code == -1
    p.run_nturn((0, 7, 3), 2)                                     # wall cell
    with pytest.raises(nhp.NhpError) as e:
        p.status()
    assert e.value.code == -4
    with pytest.raises(nhp.NhpError) as e:
        p.extract_path(sc.goal)
    assert e.value.code == -4
    assert (p.cost_volume_numpy() == INF).all()
    p.run_nturn(sc.start, 3)
    p.status()
    assert p.extract_path(sc.start) == ([tuple(sc.start) + (-1,)], 0)
    with pytest.raises(nhp.NhpError) as e:
        p.extract_path((0, 5, 5))
    assert e.value.code == -5
    x, y, th = p.index_to_pose(*sc.start)
    assert p.pose_to_index(x, y, th) == tuple(sc.start)
    # empty obstacle image and an all-blocked image
    p.render_obstacles(np.zeros_like(sc.hard))
    p.run_nturn(sc.start, 2)
    V = p.cost_volume_numpy()
    assert (V[:, 0, :] == INF).all() and (V[:, :, 0] == INF).all() and (V != INF).sum() > 0.5 * V.size
    p.render_obstacles(np.ones_like(sc.hard))
    assert p.collision_numpy().all()
    p.close()
    with pytest.raises(nhp.NhpError) as e:
        nhp.Planner(9, 8, 80.0, sc.ct)                            # N_theta < 2 pi R
    assert e.value.code == -3


def _sweeps_match(mods, sc, flags, n_cycles):
    oracle, nhp = mods
    o, fp = oracle_for(oracle, sc, threads=0)
    p = nhp.Planner.from_scene(sc, flags=flags)
    p.render_obstacles(sc.hard, sc.soft)
    Cv, Sv = o.render(fp, sc.hard, sc.soft, method="runs")
    assert (p.collision_numpy() == Cv).all()
    p.run_nturn(sc.start, n_cycles)
    got = p.cost_volume_numpy()
    V = o.run(Cv, Sv, sc.start, n_cycles)
    assert (got == V).all(), (sc.name, flags, int((got != V).sum()))
    assert (V != INF).any()
    p.close()


def test_straight_sections_and_streaming_at_the_other_sizes(mods):
    """The two forms of the straight sweeps (Sections, appendix D, default up to 256 cells; streaming kernels,
    default from 512 cells) each at the sizes where they are not the default, and the extremes: one tile per line (N = 32),
    sixteen sections per line (N = 512, hard and soft), 64 tiles per line (N = 2048)."""
    oracle, nhp = mods
    _sweeps_match(mods, scenes.random_scene(5, 6, 4, 21, n_cycles=2), 0, 2)                                  # N = 32: one section
    _sweeps_match(mods, scenes.random_scene(5, 6, 4, 21, n_cycles=2), nhp.FLAG_NO_SECTIONS, 2)
    _sweeps_match(mods, scenes.get_config(3), nhp.FLAG_SECTIONS, 3)                                          # N = 512: 16 sections
    _sweeps_match(mods, scenes.get_config(4), nhp.FLAG_SECTIONS, 2)                                          # ... with soft costs
    _sweeps_match(mods, scenes.get_config(3), nhp.FLAG_SECTIONS | nhp.FLAG_FIXED_WORK, 1)
    _sweeps_match(mods, scenes.random_scene(11, 6, 8, 22, vehicle=(9, 4), n_rects=60, n_cycles=1), 0, 1)     # N = 2048: streaming
    _sweeps_match(mods, scenes.random_scene(5, 11, 6, 23, n_cycles=1), 0, 2)                                 # N_theta = 2048: turn sweeps
                                                                                                             # by the thread-per-curve kernels


def test_no_write_outside_the_buffers_and_run_to_run_identical(mods):
    """Stand-in for the memory / race checker (compute-sanitizer is closed on this pool, profiles/r02_sanitizer.md): every buffer
    handed to the library lies between guard bands that must stay untouched through footprint, rendering, both planners, every
    kernel variant and back-tracking; and the same plan run five times gives the same volume bit for bit (no two
    threads of a maneuver kernel touch the same vertex, so nothing may depend on scheduling)."""
    oracle, nhp = mods
    for sc, flags in ((scenes.random_scene(6, 6, 8, 31, soft=True, reverse_mult=512, vehicle=(5, 2), n_rects=10), 0),
                      (scenes.random_scene(6, 6, 8, 31, soft=True, reverse_mult=512, vehicle=(5, 2), n_rects=10), nhp.FLAG_NO_SECTIONS | nhp.FLAG_FIXED_WORK),
                      (scenes.random_scene(5, 10, 6, 32, n_cycles=2), 0),                    # N_theta = 1024: 32 sections per turn tile
                      (scenes.random_scene(8, 5, 4.5, 33, vehicle=(3, 2), n_rects=40, n_cycles=2), nhp.FLAG_SIMPLE_KERNELS),
                      (scenes.random_scene(7, 6, 9, 34, flags=1, soft=True), nhp.FLAG_NO_SHORTCUTS),  # forward only
                      (scenes.get_config(2), 0), (scenes.get_config(3), nhp.FLAG_SECTIONS)):
        p = nhp.Planner.from_scene(sc, flags=flags, guard_bytes=1 << 16, reach_levels=4)
        vols = []
        for rep in range(5 if sc.n <= 256 else 2):
            p.render_obstacles(sc.hard, sc.soft)
            p.run_nturn(sc.start, sc.n_cycles)
            vols.append(p.cost_volume().clone())
            try:
                p.extract_path(sc.goal)
            except nhp.NhpError as e:
                assert e.code == -5
        assert all(bool((v == vols[0]).all()) for v in vols[1:]), sc.name
        p.reach_run(sc.start, 4)
        p.reach_count_numpy()
        assert p.guards_intact(), (sc.name, flags)
        p.close()


def test_first_cycle_with_the_sparse_launches(mods):
    """The first LF of a plan is launched as one tile and the first SF as one band per slice (sweep.cu: launch_cycles).  On small grids
    that path is taken only while the CUDA graph of the inner cycle is off, i.e. under per-kernel profiling: parity cycle by cycle
    there, for several starts, hard and soft."""
    oracle, nhp = mods
    for sc in (scenes.random_scene(6, 6, 8, 41, n_rects=8), scenes.random_scene(7, 6, 9, 42, soft=True, reverse_mult=300, vehicle=(6, 3)),
               scenes.random_scene(5, 7, 4, 43)):
        o, fp = oracle_for(oracle, sc)
        Cv, Sv = o.render(fp, sc.hard, sc.soft)
        p = nhp.Planner.from_scene(sc)
        p.render_obstacles(sc.hard, sc.soft)
        p.set_profiling(True)
        free = np.argwhere(Cv == 0)
        rng = np.random.default_rng(7)
        for k in rng.integers(len(free), size=6):
            start = (int(free[k][2]), int(free[k][1]), int(free[k][0]))
            for n_cycles in (1, 2):
                p.run_nturn(start, n_cycles)
                V = o.run(Cv, Sv, start, n_cycles)
                got = p.cost_volume_numpy()
                assert (got == V).all(), (sc.name, start, n_cycles, int((got != V).sum()))
        p.close()


def test_lane_penalty_small_scenes(mods):
    """nhp_set_lane_penalty (area / orientation penalty, DESIGN R28): the soft volume with the penalty
    folded in, the sweeps over it and the plans are the oracle's, bit for bit; host and device lane maps; through both render
    calls; switching it off restores the plain volume; N_theta below, at and above 256 (the heading is taken in 1/256 turns)."""
    oracle, nhp = mods
    import torch
    cases = [scenes.random_scene(5, 5, 4, 61, soft=True, reverse_mult=512), scenes.random_scene(6, 6, 8, 62, vehicle=(6, 3), soft=True),
             scenes.random_scene(7, 8, 9, 63, vehicle=(9, 4), n_rects=20, soft=True, n_cycles=2),
             scenes.random_scene(5, 10, 6, 64, soft=True, n_cycles=2)]
    for k, sc in enumerate(cases):
        lane_dir, lane_pen = scenes.random_lane_map(sc.n, 100 + k)
        o, fp = oracle_for(oracle, sc)
        Cv, S0 = o.render(fp, sc.hard, sc.soft, method="brute")
        S1 = o.apply_lane(S0.copy(), lane_dir, lane_pen)
        assert (S1 != S0).any()
        p = nhp.Planner.from_scene(sc)
        if k % 2:
            p.set_lane_penalty(torch.from_numpy(lane_dir).to(p.device), torch.from_numpy(lane_pen).to(p.device))
        else:
            p.set_lane_penalty(lane_dir, lane_pen)
        p.render_obstacles(sc.hard, sc.soft)
        assert (p.collision_numpy() == Cv).all() and (p.soft_numpy() == S1).all(), sc.name
        p.run_nturn(sc.start, sc.n_cycles)
        V = o.run(Cv, S1, sc.start, sc.n_cycles)
        assert (p.cost_volume_numpy() == V).all(), sc.name
        tj, jj, ij = np.nonzero(V != INF)
        rng = np.random.default_rng(k)
        for g in rng.integers(len(tj), size=10):
            goal = (int(ij[g]), int(jj[g]), int(tj[g]))
            assert p.extract_path(goal) == o.backtrack(V, Cv, S1, sc.start, goal), (sc.name, goal)
        # the device distance transform path renders with the same epilogue
        _, _, soft_dt = oracle.soft_from_hard(sc.hard, 4.0)
        _, Sdt = o.render(fp, sc.hard, soft_dt, method="brute")
        p.render_obstacles_dt(sc.hard, 4.0)
        assert (p.soft_numpy() == o.apply_lane(Sdt.copy(), lane_dir, lane_pen)).all(), sc.name
        # off again
        p.set_lane_penalty(None, None)
        p.render_obstacles(sc.hard, sc.soft)
        assert (p.soft_numpy() == S0).all(), sc.name
        with pytest.raises(nhp.NhpError) as e:
            p._check(p._L.nhp_set_lane_penalty(p._h, lane_dir.ctypes.data, None, 0), "set_lane_penalty")
        assert e.value.code == -1
        p.close()
    sc = scenes.random_scene(5, 5, 4, 1)                      # no soft volume: refused
    p = nhp.Planner.from_scene(sc)
    with pytest.raises(nhp.NhpError) as e:
        p.set_lane_penalty(*scenes.random_lane_map(sc.n, 1))
    assert e.value.code == -1
    p.close()


@pytest.mark.slow
def test_lane_penalty_two_lane_road_512(mods):
    """A 512^3 scene shaped like Figure 19: two lanes, wrong-way factor 4, centre strip 1.5.  Soft volume, cost
    volume and plans against the oracle; and what the penalty is for: goals down the start's own lane cost what they cost
    without it, the goal in the opposite lane (a U-turn) costs more."""
    oracle, nhp = mods
    sc, lane_dir, lane_pen = scenes.two_lane_road(9, 9)
    o, fp = oracle_for(oracle, sc, threads=0)
    Cv, S0 = o.render(fp, sc.hard, sc.soft, method="runs")
    S1 = o.apply_lane(S0.copy(), lane_dir, lane_pen)
    p = nhp.Planner.from_scene(sc)
    p.render_obstacles(sc.hard, sc.soft)
    p.run_nturn(sc.start, sc.n_cycles)
    V0 = p.cost_volume_numpy().copy()
    p.set_lane_penalty(lane_dir, lane_pen)
    p.render_obstacles(sc.hard, sc.soft)
    assert (p.collision_numpy() == Cv).all() and (p.soft_numpy() == S1).all()
    p.run_nturn(sc.start, sc.n_cycles)
    p.status()
    V = o.run(Cv, S1, sc.start, sc.n_cycles)
    got = p.cost_volume_numpy()
    assert (got == V).all(), int((got != V).sum())
    for goal in [sc.goal] + sc.extra_goals:
        assert p.extract_path(goal) == o.backtrack(V, Cv, S1, sc.start, goal), goal
    same_lane = [g for g in sc.extra_goals if g[2] == 0][:-1]          # the last one sits next to the end wall (soft costs differ there)
    assert all(V[g[2], g[1], g[0]] == V0[g[2], g[1], g[0]] for g in same_lane)
    g = sc.goal
    assert V[g[2], g[1], g[0]] > V0[g[2], g[1], g[0]]
    p.close()


@pytest.mark.slow
def test_sparse_first_cycle_at_512_as_production_runs_it(mods):
    """At 512^3 no CUDA graph is in use, so the one-tile first LF and the one-band-per-slice first SF are what every plan runs
    (no profiling needed).  Starts are chosen so that the branches of those launches are all taken: a left-turn tile that wraps
    the seam in x (tile column 0 and the last one) and one that does not, a start whose straight line lies in the last band of a
    slice swept along x (I = 0) and of one swept along y (I = 1), a start on a diagonal heading, and random ones; hard (config 3)
    and soft (config 4).  One cycle and two, whole volume."""
    oracle, nhp = mods
    for cfg, n_random in ((3, 2), (4, 1)):
        sc = scenes.get_config(cfg)
        o, fp = oracle_for(oracle, sc, threads=0)
        Cv, Sv = o.render(fp, sc.hard, sc.soft, method="runs")
        p = nhp.Planner.from_scene(sc)
        assert p.cycle_graph_kernels() == 0
        p.render_obstacles(sc.hard, sc.soft)
        n, nt, mx, q = sc.n, sc.nt, sc.n - 1, sc.nt // 4
        beta, B, I = o.beta.astype(np.int64), o.B.astype(np.int64), o.I
        rng = np.random.default_rng(cfg)
        flat = rng.integers(Cv.size, size=2000000)
        flat = flat[Cv.reshape(-1)[flat] == 0]                           # free poses
        tt, jj, ii = flat // (n * n), (flat // n) % n, flat % n
        tile = ((ii - beta[tt]) & mx) >> 5                               # eq (18) inverted: tile column of the left-turn curve through the start
        line = np.where(I[tt] == 0, (jj - B[tt, ii]) & mx, (ii - B[tt, jj]) & mx) >> 5      # eq (23) inverted: band of the straight line
        wanted = [("tile column 0", tile == 0), ("last tile column", tile == n // 32 - 1), ("inner tile column", tile == n // 64),
                  ("last band, I = 0", (line == n // 32 - 1) & (I[tt] == 0)), ("last band, I = 1", (line == n // 32 - 1) & (I[tt] == 1)),
                  ("diagonal heading", tt % (nt // 8) == 0)] + [("random", np.ones(len(tt), bool))] * n_random
        if cfg == 4:
            wanted = wanted[::2]
        for what, ok in wanted:
            k = np.flatnonzero(ok)
            assert len(k), what
            k = k[rng.integers(len(k))]
            start = (int(ii[k]), int(jj[k]), int(tt[k]))
            for n_cycles in ((1, 2) if what in ("tile column 0", "last band, I = 1") else (1,)):
                p.run_nturn(start, n_cycles)
                p.status()
                V = o.run(Cv, Sv, start, n_cycles)
                got = p.cost_volume_numpy()
                assert (got == V).all(), (sc.name, what, start, n_cycles, int((got != V).sum()))
        p.close()


def _full_config(mods, k, sample_render=20000):
    oracle, nhp = mods
    sc = scenes.get_config(k)
    o, fp = oracle_for(oracle, sc, threads=0)
    p = nhp.Planner.from_scene(sc)
    p.render_obstacles(sc.hard, sc.soft)
    Cg, Sg = p.collision_numpy(), p.soft_numpy()
    # rendering: sampled poses against the brute-force definition, then the whole volume against the run renderer
    rng = np.random.default_rng(k)
    for _ in range(sample_render if sc.n <= 256 else sample_render // 10):
        i, j, t = int(rng.integers(sc.n)), int(rng.integers(sc.n)), int(rng.integers(sc.nt))
        c, s = o.render_pose(fp, sc.hard, sc.soft, i, j, t)
        assert c == Cg[t, j, i] and (Sg is None or s == Sg[t, j, i]), (i, j, t)
    # whole volume: against the plain O(N_R |box|) loop where that takes seconds (configs 1 and 2), else against the run-decomposed
    # renderer (itself pinned to the plain loop in tests/test_oracle_render.py, incl. the footprint of config 5)
    Cv, Sv = o.render(fp, sc.hard, sc.soft, method="brute" if sc.n <= 256 else "runs")
    assert (Cg == Cv).all()
    if Sv is not None:
        assert (Sg == Sv).all()
    del Cg, Sg
    if sc.n > 256:
        # three whole Theta planes by the plain per-pose loop as well: an axis heading, a diagonal, a generic angle
        for t in (0, sc.nt // 8, (5 * sc.nt) // 13 | 1)[(1 if sc.n > 512 else 0):]:      # config 5: seconds per plane, two planes
            Cp, Sp = o.render_plane(fp, sc.hard, sc.soft, t)
            assert (Cp == Cv[t]).all(), t
            assert Sv is None or (Sp == Sv[t]).all(), t
    p.run_nturn(sc.start, sc.n_cycles)
    p.status()
    got = p.cost_volume_numpy()
    V = o.run(Cv, Sv, sc.start, sc.n_cycles)
    assert (got == V).all(), int((got != V).sum())
    goals = [sc.goal] + list(sc.extra_goals[:: max(1, len(sc.extra_goals) // 16)])
    reached = 0
    for goal in goals:
        try:
            want = o.backtrack(V, Cv, Sv, sc.start, goal)
            reached += 1
        except oracle.OracleError as e:
            with pytest.raises(nhp.NhpError) as g:
                p.extract_path(goal)
            assert g.value.code == e.code
            continue
        assert p.extract_path(goal) == want, goal
    p.close()
    return reached, float((V != INF).mean())


def test_config1_rects_64(mods):
    reached, frac = _full_config(mods, 1)
    assert reached == 1 and frac > 0.2


def test_config2_parallel_parking_256(mods):
    reached, frac = _full_config(mods, 2)
    assert reached == 1


@pytest.mark.slow
def test_config3_maze_512(mods):
    reached, frac = _full_config(mods, 3)
    assert reached >= 3


@pytest.mark.slow
def test_config4_cluttered_512(mods):
    reached, frac = _full_config(mods, 4)
    assert reached == 1


@pytest.mark.slow
def test_config5_perpendicular_lot_1024(mods):
    reached, frac = _full_config(mods, 5)
    assert reached == 1
