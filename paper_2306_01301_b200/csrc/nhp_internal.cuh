// Internal declarations of libnhplan.so (CUDA path).  Shares nothing with oracle/.
// Citations: PAPER.md = /root/reference/PAPER.md; DESIGN R<k> = readings in /root/repo/DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/nhplan.h"

// ---- internal value encoding of the volume V while sweeps run -------------
//   0            vertex is blocked (stamped from the collision bits by the init kernel)
//   1 .. 2^30    cost + 1 of a reached vertex
//   VI_INF       free vertex not reached yet
// Any in-register value >= VI_INF means "infinite"; min(arrival, stored) therefore never needs a
// clamp: blocked cells keep 0, unreached cells keep VI_INF, and nothing above VI_INF is ever stored.
constexpr uint32_t VI_INF = (1u << 30) + 1u;
constexpr uint32_t VI_BIG = VI_INF;            // added on edges that leave a blocked vertex

enum { M_LF = 0, M_SF = 1, M_RB = 2, M_RF = 3, M_SB = 4, M_LB = 5 };

#ifdef __CUDACC__
// One vertex of a maneuver sweep, exactly the paper's line (Insert 5) in the internal encoding:
//     v <- min(v, u + ct) + cx * B[i]              (arriving value v, stored value u, edge weight w at the SOURCE vertex)
// with "infinity" leaving a blocked vertex (u == 0; blocked vertices are removed, DESIGN R10).
// Three instructions, two of them on the min/max (DPX) pipe:
//     e  = u + ct + w
//     x  = min(v + w, e)                           unsigned: v <= 2^31 - 1 and w < 2^26, no wrap
//     v' = max_signed(u + 0x7fffffff, x)           u == 0 -> INT_MAX ("infinite"); u >= 1 wraps negative -> x
// Every value >= VI_INF is "infinite"; x < 2^31 because e < 2^31.
__device__ __forceinline__ uint32_t nhp_chain_step(uint32_t v, uint32_t u, uint32_t w, uint32_t ct)
{
    const uint32_t e = u + ct + w;
    const uint32_t x = __viaddmin_u32(v, w, e);
    return (uint32_t)__viaddmax_s32((int)u, 0x7fffffff, (int)x);
}

// The same line with the arriving value carried as a = v - ct ("transition cost not charged yet") and the edge weight
// of the PREVIOUS vertex still pending: t = min(a, u) is the value at the vertex before its own edge, so
//     t_k   = min(t_{k-1} + w_{k-1}, u_k)                           one DPX op, no separate addition
//     out_k = min(v_k, u_k) = min(t_k + ct, u_k)                    one DPX op (u_k <= u_k + ct)
//     t_k  <- "infinite" if the vertex is blocked (u_k == 0)        one DPX op (signed max against u + INT_MAX)
// a never goes negative: every finite v is some u_j + ct + (edge weights) >= 1 + ct.  No wrap: t <= 2^31 - 1,
// w, ct < 2^26.  Identical integers to nhp_chain_step (a + ct = v), two / three ALU ops per vertex instead of
// three / four.
__device__ __forceinline__ uint32_t nhp_arrive(uint32_t t_prev, uint32_t w_prev, uint32_t u)
{
    return __viaddmin_u32(t_prev, w_prev, u);
}
__device__ __forceinline__ uint32_t nhp_keep(uint32_t t, uint32_t ct, uint32_t u)
{
    return __viaddmin_u32(t, ct, u);
}
__device__ __forceinline__ uint32_t nhp_gate(uint32_t t, uint32_t u)
{
    return (uint32_t)__viaddmax_s32((int)u, 0x7fffffff, (int)t);
}

// Soft edge weight (len_q * S) >> 4 (DESIGN R18) from len4 = len_q << 4 and byte `b` of a word of four S values:
// one PRMT (S << 24) and one IMAD.HI.
__device__ __forceinline__ uint32_t nhp_soft_weight(uint32_t len4, uint32_t packed, int b)
{
    return __umulhi(len4, __byte_perm(packed, 0u, (uint32_t)((b << 12) | 0x444)));
}
#endif

struct DevTables {
    const int16_t *beta;    // [nt]      beta(Theta), eq (13)-(17) PAPER.md:233-262
    const int16_t *B;       // [nt][n]   B(y',Theta) = round(y' K(Theta))
    const uint32_t *len_q;  // [6][nt]   fixed-point edge length
    const uint8_t *IJ;      // [nt]      bit0 = I(Theta) eq (19), bit1 = (J(Theta) > 0) eq (24)
};

struct nhp_planner {
    int log2_n = 0, log2_nt = 0, n = 0, nt = 0;
    double R = 0;
    nhp_weights w{};
    nhp_limits lim{};              // resolved limits (defaults filled in)
    int device = 0;                // ordinal of the device that owns the caller's buffers; current inside every call
    cudaStream_t stream = nullptr;
    uint32_t *V = nullptr, *C = nullptr;
    uint8_t *S = nullptr;
    uint8_t *S_left = nullptr, *S_right = nullptr, *S_line = nullptr;   // curve-major copies of S (workspace), soft only
    // host tables (fp64 once, then integers)
    std::vector<int32_t> beta, B, cosq, sinq;
    std::vector<uint8_t> psi2, I;
    std::vector<int8_t> J;
    std::vector<uint32_t> len_q;
    // device tables (library-owned, small)
    int16_t *d_beta = nullptr, *d_B = nullptr;
    uint32_t *d_lenq = nullptr;
    uint8_t *d_IJ = nullptr;
    int16_t *d_tlist = nullptr;    // [nt] slices with I = 0 first (n_xslices of them), then those with I = 1
    int n_xslices = 0;
    uint32_t *d_xl_tab = nullptr;  // [n_xslices][n/32][32] tile word of every lane of the x-rows kernel (straight.cu: straight_xl_kernel)
    int32_t *d_rot = nullptr;      // [nt][4] cosq, sinq, 2*Psi0, 2*Psi1
    // footprint (all in the caller's workspace, sized for lim.max_footprint_radius)
    int rad = 0, side = 0, sidew = 0;
    uint8_t *d_mask = nullptr;     // [(2 rmax + 1)^2]
    uint32_t *d_E = nullptr;       // [nt][side][sidew] bitmap of covered pixel offsets, bit (da + rad)
    size_t cap_runs = 0;           // capacity of d_runs, entries
    int cap_levels = 1;            // capacity of d_Hk / d_Mk, levels
    bool have_footprint = false;
    // images
    uint8_t *d_hard = nullptr, *d_soft = nullptr;
    uint8_t *d_lane_dir = nullptr, *d_lane_pen = nullptr;   // [n][n] lane map of nhp_set_lane_penalty (DESIGN R28), soft planners only
    bool have_lane = false;
    int32_t *d_dtg = nullptr;      // [n][n] column distances of the distance transform (distance.cu), soft planners only
    // run decomposition of E_Theta and the sparse tables of the image rows (render.cu)
    int4 *d_runs = nullptr;        // (db, da_lo, second look-up offset, level) of every run, grouped by Theta
    int32_t *d_run_off = nullptr;  // [nt + 1] first run of every Theta
    int n_levels = 1, max_runs = 0;
    uint32_t *d_Hk = nullptr;      // [levels][n][n/32] hard | wall, bit-packed rows; level k = OR over 2^k columns
    uint8_t *d_Mk = nullptr;       // [levels][n][n]    soft image; level k = max over 2^k columns (soft only)
    bool have_render = false, have_run = false, canonical = false;
    int start[3] = {0, 0, 0};
    // reachability (bit-vector) planner, reach.cu: level volumes and the transposed working volumes (carved from the caller's
    // workspace at create), number of levels of the last run, its start
    uint32_t *r_levels = nullptr, *r_Lt = nullptr, *r_Ct = nullptr, *r_Gt = nullptr;   // in the caller's workspace
    int r_n_levels = -1, r_start[3] = {0, 0, 0};
    int sparse_xp = -1, sparse_yp = -1;   // >= 0 only while launch_cycles launches the first SF of a plan (straight.cu: StartCurve)
    int start_m0 = -1;             // maneuver in progress at the start (nhp_run_nturn_from), -1 = none
    // plan extraction
    int32_t *d_status = nullptr;   // N-turn planner: [0] start blocked, [1] backtrack rc, [2] count, [3] cost, [4..7] goal search:
                                   // i, j, theta, goal index, [8..9] its score, [10] found; NHP_STATUS_WORDS words.  The plan
                                   // follows directly (d_plan = d_status + NHP_STATUS_WORDS): one copy brings both back
    int32_t *d_rstatus = nullptr;  // reachability planner: its own [0] start blocked, [1] rc, [2] count, [3] maneuvers, then its plan
    int32_t *d_goals = nullptr;    // [NHP_MAX_GOALS][3] ideal goals of nhp_extract_path_goalset
    nhp_waypoint *d_plan = nullptr, *d_rplan = nullptr;
    int plan_cap = 0, plan_eager = 128;    // waypoints brought back together with the status words (NHP_PLAN_EAGER)
    int32_t *h_status = nullptr;   // pinned: NHP_STATUS_WORDS words, then plan_cap waypoints
    nhp_waypoint *h_plan = nullptr;
    // CUDA graph of one inner maneuver cycle (sweep.cu: build_cycle_graph), instantiated at creation for grids small enough
    // for the launch overhead to matter; replayed by launch_cycles unless per-kernel profiling is on
    cudaGraph_t cycle_graph = nullptr;
    cudaGraphExec_t cycle_exec = nullptr;
    int cycle_graph_kernels = 0;
    std::string err = "ok";
    long long launches = 0;
    // per-kernel timing (nhp_set_profiling): event pairs on the launching stream, drained at sync points
    bool profiling = false;
    std::vector<cudaEvent_t> ev;   // 2 events per pair; the pool grows by PROF_GROW pairs when it runs out, up to PROF_MAX_PAIRS
    std::vector<int> ev_slot;      // slot of each used pair
    int ev_used = 0;
    long long ev_dropped = 0;      // launches that ran untimed because the pool was at its maximum
    double k_ms[NHP_KERNEL_SLOTS] = {0};
    long long k_launches[NHP_KERNEL_SLOTS] = {0};

    DevTables tables() const { return DevTables{d_beta, d_B, d_lenq, d_IJ}; }
};

constexpr int PROF_GROW = 1024, PROF_MAX_PAIRS = 65536;
constexpr int NHP_STATUS_WORDS = 16;
constexpr int NHP_MAX_GOALS = 256;
constexpr int NHP_PLAN_CAP = 4096;         // waypoints of the internal plan buffers

bool prof_grow(nhp_planner *p);            // api.cu: add PROF_GROW event pairs; false at the maximum or on a CUDA error

// Makes the handle's device current for the duration of an ABI call (the caller may have another one current).
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const nhp_planner *p)
    {
        if (!p) return;
        int cur = -1;
        if (cudaGetDevice(&cur) == cudaSuccess && cur != p->device) { prev = cur; cudaSetDevice(p->device); }
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Bracket one kernel launch (or one group of launches) with an event pair when profiling is on.
struct ProfScope {
    nhp_planner *p;
    int pair;
    ProfScope(nhp_planner *p_, int slot) : p(p_), pair(-1)
    {
        if (!p->profiling) return;
        if (2 * (size_t)p->ev_used >= p->ev.size() && !prof_grow(p)) { p->ev_dropped++; return; }
        pair = p->ev_used++;
        p->ev_slot[pair] = slot;
        cudaEventRecord(p->ev[2 * pair], p->stream);
    }
    ~ProfScope()
    {
        if (pair >= 0) cudaEventRecord(p->ev[2 * pair + 1], p->stream);
    }
};

// ---- kernel launchers (each returns the number of kernels it launched) ---------------------------
int launch_footprint_raster(nhp_planner *p, int mw, int mh, int64_t ouq, int64_t ovq);
int finish_footprint(nhp_planner *p);                 // host: run lists into the workspace tables; returns an NHP_ code
int launch_render(nhp_planner *p, bool soft);
int launch_init_volume(nhp_planner *p, int si, int sj, int st);
int launch_export_volume(nhp_planner *p, bool to_canonical);
int launch_cycles(nhp_planner *p, int n_cycles, bool fresh);   // fresh: the volume has just been initialised (one finite vertex)
int build_cycle_graph(nhp_planner *p);               // at creation; NHP_OK also when no graph is built
int launch_backtrack(nhp_planner *p, int gi, int gj, int gt);     // gi < 0: the goal comes from launch_goal_search
int launch_goal_search(nhp_planner *p, int n_goals, int d, uint32_t W, uint32_t w);
int launch_seed_in_progress(nhp_planner *p, int m0);
int launch_reach_run(nhp_planner *p, int si, int sj, int st, int n_levels, int *launches);   // reach.cu
int launch_reach_backtrack(nhp_planner *p, int gi, int gj, int gt);
int launch_reach_count(nhp_planner *p, uint8_t *K_dev);
int launch_straight_tile(nhp_planner *p, int m);      // straight.cu; 0 = not applicable
int launch_soft_layouts(nhp_planner *p);
int launch_soft_from_hard(nhp_planner *p, float k, float *dist_dev, int32_t *d2_dev);   // distance.cu: d_hard -> d_soft              // softlayout.cu: S -> S_left, S_right, S_line
