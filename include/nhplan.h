/*
 * nhplan.h -- C ABI of libnhplan.so: the kernel-style N-turn planner of
 * "Nonholonomic Motion Planning as Efficient as Piano Mover's" (arXiv 2306.01301) on one B200.
 *
 * Citations are lines of /root/reference/PAPER.md ("PAPER.md:<line>", with section / equation);
 * "DESIGN R<k>" is a numbered reading in /root/repo/DESIGN.md section 3.
 *
 * The pipeline behind these calls is the paper's 8-step algorithm (section XI):
 *   obstacle image -> [nhp_render_obstacles: steps 3-4] -> [nhp_run_nturn: step 5]
 *   -> [nhp_extract_path: steps 6-8] -> plan on the host.
 * Every step runs in hand-written CUDA kernels for sm_100a; there is no CPU fallback.  The library
 * allocates device memory in nhp_planner_create only ("no memory allocation takes place during processing",
 * PAPER.md:565): the large buffers are the caller's (nhp_buffers, sized by nhp_query_sizes from the grid and the
 * nhp_limits), the small tables are the library's.  All work is enqueued on the caller's stream; only the
 * nhp_extract_path family, nhp_render_vehicle_footprint, nhp_status, nhp_kernel_times and the debug accessors
 * synchronise that stream.  Every entry point makes the handle's device current for the duration of the call.
 *
 * Grid: N x N spatial cells (N = 2^log2_n) and N_theta = 2^log2_ntheta headings,
 * Theta <-> angle 2 pi Theta / N_theta, all indices taken modulo their dimension, one-cell hard wall
 * at i = 0 and j = 0.  Volume index idx = (Theta * N + j) * N + i  (i = x fastest).
 * Vertex (i, j, Theta) stands for the pose (i + Psi0(Theta), j + Psi1(Theta), theta(Theta)), eq (16) l.256.
 *
 * Maneuver ids, in the paper's cycle order:
 *   0 LF left-forward, 1 SF straight-forward, 2 RB right-backward,
 *   3 RF right-forward, 4 SB straight-backward, 5 LB left-backward.
 *
 * Costs (DESIGN R18): uint32 fixed point, unit = 2^-cost_one_log2 cell of travel.  A finite cost is
 * < NHP_COST_LIMIT = 2^30; a sum that reaches the limit saturates to NHP_INF.  Blocked and unreached
 * vertices read NHP_INF in the exported volume.
 *
 * Thread safety: one handle <-> one stream <-> one caller thread at a time.
 * Memory kinds: the nhp_buffers must be plain device memory (cudaMalloc or a pool built on it) of ONE device; managed
 * (cudaMallocManaged) and host-mapped memory are refused at create with NHP_E_BUFFER, as are buffers on different devices.
 * The stream must belong to that device (not checked).
 */
#ifndef NHPLAN_H
#define NHPLAN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NHP_INF 0xFFFFFFFFu
#define NHP_COST_LIMIT (1u << 30)

/* flags of nhp_weights.flags */
#define NHP_FLAG_FORWARD_ONLY 1   /* Dubins car: only LF, SF, RF are swept */
#define NHP_FLAG_SOFT 2           /* a soft-cost volume S is rendered and used */
#define NHP_FLAG_SIMPLE_KERNELS 4 /* thread-per-curve bring-up kernels (the paper's own mapping, l.356);
                                     same results, kept for A/B measurements */
#define NHP_FLAG_FIXED_WORK 8     /* switch off the data-dependent short cuts of the sweeps (warps whose vertices are all
                                     blocked / hold no finite value yet skip their chains): every launch then executes
                                     the same instructions whatever the scene holds ("run time independent of scene",
                                     PAPER.md:39, l.565) AND stores every vertex it visits, as the paper's loop does
                                     (V[i] = min(v, u) unconditionally, Insert 5 l.948): same instructions and same bytes.
                                     Same results; for measuring the fixed-work time */
#define NHP_FLAG_SECTIONS 32      /* straight sweeps by Sections (appendix D: one warp per 32-step section of a line, all
                                     sections of a line at once, summary / ripple / apply) also on grids of more than 256 cells per side,
                                     where the streaming kernels are the default (at most 512 cells: 16 sections).  Same results */
#define NHP_FLAG_NO_SECTIONS 64   /* straight sweeps by the streaming kernels (one warp walks a whole band of lines) also on grids of at most
                                     256 cells per side, where Sections are the default.  Same results */
#define NHP_FLAG_NO_SHORTCUTS 16  /* only the first half of NHP_FLAG_FIXED_WORK: every warp runs every pass of every sweep, but a
                                     vertex is still written back only where its value improved.  Same results */

#define NHP_DEFAULT_CYCLES 8      /* PAPER.md:392 "our default is 8 cycles" (n_cycles <= 0 selects it) */

/* error codes (all entry points return 0 on success) */
#define NHP_OK 0
#define NHP_E_ARG (-1)            /* NULL / out-of-range argument */
#define NHP_E_NOT_POW2 (-2)       /* log2 sizes outside [5, 12] x [5, 12] */
#define NHP_E_ANGRES (-3)         /* N_theta < 2 pi R (DESIGN R23) */
#define NHP_E_START_BLOCKED (-4)  /* the start vertex collides */
#define NHP_E_GOAL_UNREACHED (-5) /* back-tracking found no finite predecessor */
#define NHP_E_BUFFER (-6)         /* caller buffer too small / missing */
#define NHP_E_CUDA (-7)           /* a CUDA call failed; see nhp_last_error */
#define NHP_E_STATE (-8)          /* call out of order (e.g. run before render) */
#define NHP_E_WEIGHTS (-9)        /* a cost weight is too large for the 2^30 cost range */

typedef struct nhp_planner nhp_planner;

/* Cost weights (DESIGN R8, R9).
 *   ct[m]       transition cost charged on ENTERING maneuver m from the transition state, cost units, < 2^26
 *   dir_mult[m] Q8.8 multiplier on the edge length of maneuver m (256 = 1.0; 512 on LB,SB,RB = "reverse x2")
 * Edge leaving vertex p under maneuver m costs (len_q[m][Theta_p] * S[p]) >> 4 with
 * len_q = round(2^cost_one_log2 * length * dir_mult / 256), length = 2 pi R / N_theta for turns and
 * 1/|cos| or 1/|sin| for straights, S[p] = 16 without NHP_FLAG_SOFT. */
typedef struct nhp_weights {
    uint32_t ct[6];
    uint32_t dir_mult[6];
    int32_t cost_one_log2;   /* 0..16, 10 is the default used by the benchmarks */
    int32_t flags;
} nhp_weights;

typedef struct nhp_sizes {
    size_t V_bytes;          /* value volume, uint32 per vertex            (one volume) */
    size_t C_bytes;          /* collision volume, 1 bit per vertex             */
    size_t S_bytes;          /* soft volume, uint8 per vertex; 0 without NHP_FLAG_SOFT  */
    size_t workspace_bytes;  /* everything else that scales with the grid or the limits: the footprint tables (E_Theta
                                bitmaps, run lists, sparse tables of the image rows), with NHP_FLAG_SOFT the curve-major
                                copies of S for the left-turn, right-turn and straight sweeps (3 N_R bytes), with
                                max_reach_levels > 0 the level volumes of the reachability planner
                                ((max_reach_levels + 4) N_R / 8 bytes)                                            */
} nhp_sizes;

/* Upper bounds fixed at creation so that nothing is allocated afterwards.  A NULL pointer or a zero field
 * selects the default. */
typedef struct nhp_limits {
    int32_t max_footprint_radius;  /* largest circumscribed radius of a vehicle mask around its origin, cells (+2 for Psi and
                                      rounding); default min(64, N/2 - 1).  nhp_render_vehicle_footprint / nhp_set_box
                                      fail with NHP_E_BUFFER beyond it */
    int32_t max_reach_levels;      /* largest n_levels of nhp_reach_run; default 0 = the reachability planner is not used
                                      (nhp_reach_run then fails with NHP_E_BUFFER) */
} nhp_limits;

/* Caller-owned DEVICE buffers (e.g. torch tensors), 256-byte aligned, alive until nhp_planner_destroy. */
typedef struct nhp_buffers {
    void *V;                 /* V_bytes */
    void *C;                 /* C_bytes: word (Theta*N + j)*N/32 + i/32, bit i%32 = vertex (i,j,Theta) collides */
    void *S;                 /* S_bytes or NULL: Q4.4 speed-reciprocal of vertex idx, >= 16 */
    void *workspace;         /* workspace_bytes (required with NHP_FLAG_SOFT) or NULL */
} nhp_buffers;

/* One transition point of a plan ("plan"): the vertex and the maneuver that ARRIVES at it
 * from the next record; the last record is the start and has m = -1. */
typedef struct nhp_waypoint {
    int32_t i, j, theta, m;
} nhp_waypoint;

/* Sizes of the caller-owned buffers for a grid and its limits (lim may be NULL).  Pure host arithmetic. */
int nhp_query_sizes(int log2_n, int log2_ntheta, int flags, const nhp_limits *lim, nhp_sizes *out);

/* ini(R, cT, Lx, Lt) of PAPER.md:1169.  Builds the integer tables of section V.C (beta, Psi, B, I, J,
 * edge lengths) on the host in fp64 once and uploads them.
 *   R_cells      minimum turn radius in cells, >= 1; N_theta >= 2 pi R is enforced
 *   lim          the limits the buffers were sized for (NULL = defaults), see nhp_limits
 *   dev          caller-owned device buffers (see nhp_buffers); S may be NULL without NHP_FLAG_SOFT
 *   cuda_stream  a cudaStream_t (0 = legacy default stream) on the device that owns dev->V; that device is made
 *                current inside every call on the handle
 * This is the only call that allocates device memory (the small tables, a few hundred KB).
 * Errors: NHP_E_ARG, NHP_E_NOT_POW2, NHP_E_ANGRES, NHP_E_WEIGHTS, NHP_E_BUFFER, NHP_E_CUDA. */
int nhp_planner_create(nhp_planner **out, int log2_n, int log2_ntheta, double R_cells,
                       const nhp_weights *w, const nhp_limits *lim, const nhp_buffers *dev, void *cuda_stream);

int nhp_planner_destroy(nhp_planner *p);

/* Static string describing the last error on this handle (never NULL). */
const char *nhp_last_error(const nhp_planner *p);

/* Vehicle shape (Figure 6 l.110: "the vehicle bounding shape can be arbitrary").
 *   mask_host  HOST array, mh rows x mw columns, non-zero = vehicle; column p runs along the vehicle's
 *              length axis u, row q along its width axis v
 *   origin_u/v mask pixel (p, q) owns the vehicle-frame unit square centred (p - origin_u, q - origin_v);
 *              the vehicle frame's origin is the centre of the rear axle
 * Rasterises, per Theta, the set E_Theta of image-pixel offsets covered by the footprint of a pose
 * (DESIGN R15: a pixel is covered iff its centre, rotated into the vehicle frame with Q14 integer
 * cos/sin, falls in a set mask pixel; the half-cell pose offset Psi of eq (16) is applied, l.259).
 * The footprint's circumscribed radius (+2) must be <= nhp_limits.max_footprint_radius and < N/2, and an arbitrary
 * mask may break into at most 4 runs per footprint row on average (the run lists live in the caller's workspace).
 * Synchronises the stream (mask_host may be freed on return).  Errors: NHP_E_ARG, NHP_E_BUFFER, NHP_E_CUDA. */
int nhp_render_vehicle_footprint(nhp_planner *p, const uint8_t *mask_host, int mw, int mh,
                                 double origin_u, double origin_v);

/* Bounding-box vehicle as in appendix G ("f, r, s: forward, reverse and sideways bounding box dimensions
 * in number of grid cells"): the rectangle u in [-r, f), v in [-s, s) around the centre of the rear axle, i.e.
 * nhp_render_vehicle_footprint with the all-ones (f + r) x 2 s mask and origin (r - 1/2, s - 1/2).
 * Errors: NHP_E_ARG, NHP_E_CUDA. */
int nhp_set_box(nhp_planner *p, int f, int r, int s);

/* Obstacle rendering, steps 3-4 of PAPER.md:390-391 (section VI l.338, appendix C l.871).
 *   hard  N x N uint8 image, row = y (j), column = x (i); non-zero = hard obstacle
 *   soft  N x N uint8 Q4.4 speed-reciprocal image (16 = 1.0) or NULL; requires NHP_FLAG_SOFT
 *   on_device  0: both pointers are HOST memory and are copied to the device on the stream (step 3);
 *              1: both are DEVICE pointers
 * Writes C (bit = footprint at that pose touches a hard pixel, or a pixel of the wall a = 0 / b = 0 with
 * toroidal image addressing, or i = 0, or j = 0) and, with soft, S = clamp(max of soft over the
 * footprint, 16, 255) (DESIGN R16).  Errors: NHP_E_ARG, NHP_E_STATE (no footprint yet), NHP_E_CUDA. */
int nhp_render_obstacles(nhp_planner *p, const uint8_t *hard, const uint8_t *soft, int on_device);

/* Area / orientation penalty ("direction and area-based velocity penalties"; "the rendering ... handles any
 * additional area and orientation related penalties", section VI l.338; Figure 19 l.463: "penalties to inform the planner not
 * to use the reverse direction lane and stay to the right").  The paper gives no formula; reading DESIGN R28:
 *   lane_dir  N x N uint8, row = y, column = x: preferred heading of the pixel in 1/256 turns (0 = +x, 64 = +y, 128 = -x)
 *   lane_pen  N x N uint8, Q4.4 factor (16 = 1.0 = no penalty; smaller values count as 16) on the reciprocal velocity of a
 *             vehicle that faces the opposite way; in between the factor grows linearly with the angle
 *   on_device 0: both are HOST memory, copied on the stream (keep them alive until the stream has passed the copy); 1: DEVICE
 * The next nhp_render_obstacles / nhp_render_obstacles_dt folds it into the soft volume: for the pose (i, j, Theta), read at the
 * pose's own pixel (i, j), h = floor(256 Theta / N_theta), delta = circular distance of h and lane_dir (0..128),
 *   f = 16 + (((lane_pen - 16) * 2 delta + 128) >> 8),      S <- min(255, (S * f + 8) >> 4)
 * with S the footprint maximum of the soft image (DESIGN R16).  It is a penalty on the vehicle's orientation (one obstacle
 * volume over position and orientation, l.338): reversing along a lane while facing the right way is priced by dir_mult, not
 * here.  Both pointers NULL: no penalty from the next render on.  Requires NHP_FLAG_SOFT (pass an all-16 soft image if there
 * are no soft obstacle costs).  Errors: NHP_E_ARG, NHP_E_CUDA. */
int nhp_set_lane_penalty(nhp_planner *p, const uint8_t *lane_dir, const uint8_t *lane_pen, int on_device);

/* Steps 1-4 of PAPER.md:388-391 with the distance transform on the DEVICE (the paper runs steps 1-2 on the CPU):
 * the soft image is synthesised from the hard image and then rendered exactly as by nhp_render_obstacles.
 * Reading DESIGN R17 of "some function of the distance" (section VII l.342): with H = hard | wall (row 0 and
 * column 0, not toroidal), d = float32 sqrt of the exact squared Euclidean distance to the nearest pixel of H,
 *     soft = clamp(rint(16 * (1 + k / (d + 1))), 16, 255)        Q4.4, float32, every operation rounded once.
 *   hard          N x N uint8 image as for nhp_render_obstacles (HOST, or DEVICE with on_device = 1)
 *   k             strength of the soft cost, 0 <= k <= 64 (4 in the benchmarks; 0 = no soft cost)
 *   dist_dev_out  DEVICE array of N x N floats that receives d, or NULL
 * Requires NHP_FLAG_SOFT.  Errors: NHP_E_ARG, NHP_E_STATE (no footprint yet), NHP_E_CUDA. */
int nhp_render_obstacles_dt(nhp_planner *p, const uint8_t *hard, int on_device, double k, float *dist_dev_out);

/* Steps 1-2 of PAPER.md:388-389 alone (distance transform + soft image, reading DESIGN R17 exactly as in
 * nhp_render_obstacles_dt), for callers that are NOT ALLOWED TO ALLOCATE DEVICE MEMORY and so cannot even own a planner
 * handle (nhp_planner_create calls cudaMalloc for its tables).  Who that is: a planning thread inside a vehicle's control
 * loop, where the memory budget is fixed and audited at start-up and a cudaMalloc -- which takes a driver-wide lock, may
 * wait for the whole device to go idle and can fail on a fragmented heap -- has no bounded latency; a plug-in living in a
 * process whose host framework has already claimed nearly all of HBM for its own pool, so that a raw cudaMalloc simply
 * fails; code running under a "no allocation after initialisation" rule of a safety process.  This call needs no handle,
 * calls no cudaMalloc / cudaFree and no library routine that allocates, neither on the device nor on the host.
 *
 * The one intermediate image of the transform (per pixel the distance to the nearest obstacle pixel of its column,
 * int32) lives in an array that is part of the library image itself: NHP_NOALLOC_MAX_N^2 x 4 bytes = 4 MiB of device
 * memory on EVERY GPU whose context loads libnhplan.so, held until the process exits whether or not this call is ever made.
 *   hard_dev      DEVICE, n x n uint8, row = y, column = x, non-zero = hard obstacle; row 0 and column 0 count as wall
 *   n             image side, 1 <= n <= NHP_NOALLOC_MAX_N (any n, not only powers of two).  A larger n is refused with
 *                 NHP_E_BUFFER and a message that names the limit: the array cannot grow
 *   k             strength of the soft cost, 0 <= k <= 64, as in nhp_render_obstacles_dt
 *   soft_dev_out  DEVICE, n x n uint8, receives the Q4.4 soft image (caller-owned, like every input and output)
 *   dist_dev_out  DEVICE, n x n float32, receives the distances, or NULL
 *   cuda_stream   a cudaStream_t of the device that owns the three buffers (0 = legacy default stream); the two kernels
 *                 are enqueued there and the call returns without waiting for them
 * The device that owns hard_dev is made current for the duration of the call; the outputs must live on the same device.
 * First call on a device: the library asks the runtime where that device keeps its copy of the array (each device has its
 * own, at its own address) and remembers the answer; later calls on that device skip this.  Make that first call during
 * start-up, before any stream capture is begun on the device.
 * Shared state: ALL calls on a device use the same array -- any stream, any thread -- and it keeps whatever the last
 * call left in it.  Nothing has to be cleared between calls (each call overwrites the n x n words it is going to read
 * before it reads them), but two calls whose kernels can run at the same time on one device (different streams without
 * an ordering between them) overwrite each other's intermediate image and produce garbage: order them yourself.
 * Errors: NHP_E_ARG (NULL pointer, n < 1, k out of range), NHP_E_BUFFER (n > NHP_NOALLOC_MAX_N; a pointer that is not
 * plain device memory or lives on another device), NHP_E_CUDA.  nhp_noalloc_last_error() returns the text of the calling
 * thread's last failure of this entry point ("" after a success; never NULL; static storage). */
#define NHP_NOALLOC_MAX_N 1024
int nhp_soft_from_hard_noalloc(const uint8_t *hard_dev, int n, double k, uint8_t *soft_dev_out, float *dist_dev_out,
                               void *cuda_stream);
const char *nhp_noalloc_last_error(void);

/* Debug accessor: the soft image the last render used (N x N uint8) -> HOST.  Synchronises the stream. */
int nhp_debug_soft_image(nhp_planner *p, uint8_t *soft_host);

/* Step 5 of PAPER.md:392: V <- INF, V[start] <- 0, then n_cycles maneuver cycles LF, SF, RB, RF, SB, LB
 * (PAPER.md:475), each an in-place min-plus sweep of every curve of that maneuver (Inserts
 * 3-5 l.922-949) gated by C and weighted by S.  n_cycles <= 0 selects the paper's default of 8.
 * A blocked start is reported by the next nhp_extract_path / nhp_status (the check runs on the device).
 * Errors: NHP_E_ARG, NHP_E_STATE, NHP_E_CUDA. */
int nhp_run_nturn(nhp_planner *p, int i, int j, int theta, int n_cycles);

/* nhp_run_nturn with a maneuver IN PROGRESS at the start (section XII: "the current maneuver state
 * should also be encoded in the graph when a plan is in progress ... if a maneuver is in progress, there should be no
 * transition cost to start with that maneuver").  Reading DESIGN R26: besides V[start] = 0, the vertices ahead of the
 * start on the curve of maneuver m0 are seeded with the summed edge weights from the start, without ct[m0], up to the
 * first blocked vertex (at most one lap); nhp_extract_path then charges no ct for the segment that leaves the start
 * under m0.  m0 = -1: no maneuver in progress (= nhp_run_nturn).  Errors as nhp_run_nturn; NHP_E_ARG for a reverse
 * maneuver with NHP_FLAG_FORWARD_ONLY. */
int nhp_run_nturn_from(nhp_planner *p, int i, int j, int theta, int m0, int n_cycles);

/* Reachability ("bit-vector") planner of appendix C: cost = number of maneuvers, one BIT per pose.
 * Level volume m holds the poses reachable from the start with <= m maneuvers (bit = 1; layout as C); level m + 1 =
 * level m OR the sweeps of all maneuvers over level m (l.871, Insert 2 l.873-878); the n_levels + 1 volumes are
 * kept for back-tracking (l.897).  Uses the collision volume of the last nhp_render_obstacles and none of the costs
 * (soft volume, ct, dir_mult); NHP_FLAG_FORWARD_ONLY is honoured.  n_levels <= 0 selects 8; at most 254.
 * The level volumes and three working volumes live in the caller's workspace: n_levels <= nhp_limits.max_reach_levels.
 * Errors: NHP_E_ARG, NHP_E_STATE, NHP_E_BUFFER, NHP_E_CUDA; a blocked start is reported by nhp_reach_extract_path. */
int nhp_reach_run(nhp_planner *p, int i, int j, int theta, int n_levels);

/* Borrowed DEVICE pointer to the level volumes of the last nhp_reach_run: level m starts at word m * N_R / 32. */
int nhp_reach_levels(nhp_planner *p, const uint32_t **dev_ptr_out, int *n_levels);

/* K[Theta][j][i] (uint8, DEVICE buffer of N_R bytes owned by the caller) = fewest maneuvers that reach the pose = the
 * first level whose bit is set; 255 = not reached within the levels of the last nhp_reach_run (or blocked). */
int nhp_reach_count_volume(nhp_planner *p, uint8_t *K_dev);

/* Back-tracking over the level volumes: from the goal at its level k, the maneuvers in cycle order; each walks back
 * along its curve until a blocked vertex and offers the first vertex reachable with <= k - 1 maneuvers; the first
 * maneuver with an offer wins (DESIGN R27).  Records as nhp_extract_path; *n_maneuvers = level of the goal.
 * Errors: NHP_E_ARG, NHP_E_STATE, NHP_E_START_BLOCKED, NHP_E_GOAL_UNREACHED, NHP_E_BUFFER, NHP_E_CUDA. */
int nhp_reach_extract_path(nhp_planner *p, int gi, int gj, int gtheta, nhp_waypoint *out_host, int cap, int *count,
                           int *n_maneuvers);

/* Continue sweeping the existing value volume for n_cycles more cycles. */
int nhp_run_more(nhp_planner *p, int n_cycles);

/* Cost-to-come volume in canonical form: uint32 [Theta][j][i], NHP_INF on blocked / unreached vertices.
 * *dev_ptr_out is the caller's own V buffer (borrowed, DEVICE), valid until the next run / destroy.  The
 * conversion from the sweeps' internal encoding is enqueued on the stream (one pass over V). */
int nhp_cost_volume(nhp_planner *p, const uint32_t **dev_ptr_out);

/* Steps 6-8 of PAPER.md:393-395 with an explicit goal vertex (DESIGN R20): repeated reverse Bellman step
 * over the six whole curves through the current vertex, eq (32) l.380; ties resolve to the earliest
 * maneuver in cycle order, then to the nearest source (DESIGN R19).
 *   out_host  HOST array of cap records, filled goal -> start
 *   count     number of records written;  cost: sum over segments of ct[m] + edge weights
 * Synchronises the stream.  Errors: NHP_E_ARG, NHP_E_STATE, NHP_E_START_BLOCKED, NHP_E_GOAL_UNREACHED,
 * NHP_E_BUFFER (plan longer than cap), NHP_E_CUDA. */
int nhp_extract_path(nhp_planner *p, int gi, int gj, int gtheta, nhp_waypoint *out_host, int cap,
                     int *count, uint32_t *cost);

/* Steps 6-8 with a goal SET and a reward (section IX: "more than one configuration in the goal
 * set and ... a reward function ... The optimization criterion is the reward for the vertex minus the cost to get
 * there ... Multiple ideal goals is also possible"; parameters d, W, w of appendix G l.1169).  Reading DESIGN R20:
 *   goal set of ideal goal g = vertices (gi+di, gj+dj, (gtheta+dt) mod N_theta), di^2 + dj^2 <= d^2, |dt| <= d,
 *   clipped at the grid border, not blocked, reached;   criterion  min  V + W (di^2 + dj^2) + w dt^2  (cost units);
 *   ties: first in the order (goal index, dt, dj, di), each ascending.
 *   goals_host  HOST array of n_goals x 3 int32 (i, j, theta), 1 <= n_goals <= 256;  0 <= d <= 31;  W, w < 2^20
 *   chosen      HOST int32[4] or NULL: the winning vertex (i, j, theta) and the index of its ideal goal
 *   score       HOST or NULL: the criterion of the winner
 * The search runs on the device ("to avoid transferring the value volume", l.374) and hands its result to the
 * back-tracking kernel without a host round trip; the plan starts at the chosen vertex.  d = 0 with one goal is
 * nhp_extract_path.  Errors as nhp_extract_path; NHP_E_GOAL_UNREACHED if no vertex of any goal set is reached. */
int nhp_extract_path_goalset(nhp_planner *p, const int32_t *goals_host, int n_goals, int d, uint32_t W, uint32_t w,
                             nhp_waypoint *out_host, int cap, int *count, uint32_t *cost, int32_t *chosen, uint64_t *score);

/* Synchronise and report device-side conditions of the last run (NHP_OK or NHP_E_START_BLOCKED). */
int nhp_status(nhp_planner *p);

/* eq (16) PAPER.md:256 and its inverse (nearest vertex). x, y in cells, theta in radians. */
int nhp_index_to_pose(const nhp_planner *p, int i, int j, int theta, double *x, double *y, double *theta_rad);
int nhp_pose_to_index(const nhp_planner *p, double x, double y, double theta_rad, int *i, int *j, int *theta);

/* Debug accessor: copies the library's tables to HOST arrays (any pointer may be NULL).
 *   beta int32[N_theta], psi2 uint8[N_theta] (= 2 Psi), B int32[N_theta][N], I uint8[N_theta],
 *   J int8[N_theta], len_q uint32[6][N_theta] */
int nhp_debug_tables(const nhp_planner *p, int32_t *beta, uint8_t *psi2, int32_t *B, uint8_t *I, int8_t *J,
                     uint32_t *len_q);

/* Debug accessor: the structuring elements E_Theta of the current footprint (DESIGN R15) -> HOST.
 *   *radius   receives rad; the elements are (2 rad + 1) x (2 rad + 1) offset windows
 *   covered   HOST uint8 [N_theta][2 rad + 1][2 rad + 1] or NULL (size query): covered[Theta][db + rad][da + rad] = 1 iff
 *             the footprint of a pose of heading Theta covers the image pixel (i + da, j + db)
 *   cap       bytes available at `covered`
 * Synchronises the stream.  Errors: NHP_E_ARG, NHP_E_STATE (no footprint yet), NHP_E_BUFFER, NHP_E_CUDA. */
int nhp_debug_footprint(nhp_planner *p, int *radius, uint8_t *covered, size_t cap);

/* Debug setter: how many waypoints of a plan come back in the same device-to-host copy as the status words (default 128; a
 * longer plan takes a second copy).  Tests set it to a small number to exercise the second copy with short plans.
 * 1 <= n_waypoints <= 4096.  Errors: NHP_E_ARG. */
int nhp_debug_set_plan_eager(nhp_planner *p, int n_waypoints);

/* Debug accessor: number of kernels in the CUDA graph of one inner maneuver cycle that nhp_run_nturn replays while profiling is
 * off (grids of at most 2^26 poses with the tile kernels), 0 if the handle launches every kernel separately. */
int nhp_debug_cycle_graph_kernels(const nhp_planner *p);

/* Number of kernels launched by this handle since creation (for bench.py's gpu_launches). */
long long nhp_launch_count(const nhp_planner *p);

/* Per-kernel device timing for bench.py's roofline line.  With profiling enabled every kernel launch of the
 * handle is bracketed by a cudaEvent pair recorded on the handle's stream (the pool of events grows as needed, up to
 * 65536 launches between two reads; launches beyond that run untimed and are counted by nhp_prof_dropped).
 * nhp_kernel_times synchronises the stream, adds the elapsed times
 * of the pairs recorded since the last read to running sums, copies the sums to HOST arrays of
 * NHP_KERNEL_SLOTS entries and, with reset != 0, zeroes them.
 *   slots 0..5  maneuver kernels in cycle order (LF, SF, RB, RF, SB, LB)
 *   slot 6      collision rendering (a1), slot 7 soft rendering (a2), slot 8 volume init / export (a6),
 *   slot 9      back-tracking (a7), slot 10 footprint rasterisation + image packing,
 *   slot 11     turn-pair launches (RB+RF or LB+next LF in one kernel: two maneuvers per launch)
 *   slot 12     distance transform + soft-image synthesis (nhp_render_obstacles_dt)
 *   slot 13     one level of the reachability planner (all its launches: copy, six sweeps, transpositions)
 *   slot 14     the I = 0 ("x-rows") kernel of a straight maneuver alone, slot 15 its I = 1 ("rows") kernel alone: both are
 *               NESTED inside the SF / SB pair of slots 1 and 4 (do not add them to a sum over the slots)
 *   slot 16     a straight maneuver in its Sections form (one launch for both slice groups), nested in the same way */
#define NHP_KERNEL_SLOTS 17
int nhp_set_profiling(nhp_planner *p, int enable);
int nhp_kernel_times(nhp_planner *p, double *ms_sum, long long *launches, int reset);
/* Launches that ran untimed since creation because the event pool was exhausted (0 in any sane use). */
long long nhp_prof_dropped(const nhp_planner *p);

#ifdef __cplusplus
}
#endif
#endif /* NHPLAN_H */
