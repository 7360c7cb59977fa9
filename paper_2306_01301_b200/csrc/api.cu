// C ABI of libnhplan.so (include/nhplan.h): argument checking, host-side table build
// and kernel launches.  No planning arithmetic runs on the host after nhp_planner_create.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "nhp_internal.cuh"

int set_kernel_attributes(nhp_planner *p);     // straight.cu: per-device function attributes, set at creation

namespace {

constexpr double kPi = 3.14159265358979323846;

int fail(nhp_planner *p, int code, const char *what)
{
    if (p) p->err = what;
    return code;
}

int cuda_fail(nhp_planner *p, cudaError_t e, const char *where)
{
    if (p) p->err = std::string(where) + ": " + cudaGetErrorString(e);
    return NHP_E_CUDA;
}

#define CU(call)                                                   \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(p, e_, #call);     \
    } while (0)

// sin(2 pi k / nt), argument reduced to the first octant in integers so that the symmetries the paper
// relies on (Psi_2 = Psi_0, Psi_3 = Psi_1; tan = +-1 exactly on the diagonals, DESIGN R5)
// hold bit for bit.
double sin_frac(int k, int nt)
{
    const int half = nt / 2, q = nt / 4;
    k &= nt - 1;
    double sign = 1.0;
    if (k >= half) { k -= half; sign = -1.0; }
    if (k > q) k = half - k;
    double s;
    if (k == 0) s = 0.0;
    else if (k == q) s = 1.0;
    else if (2 * k <= q) s = std::sin(2.0 * kPi * (double)k / (double)nt);
    else s = std::cos(2.0 * kPi * (double)(q - k) / (double)nt);
    return sign * s;
}

// Section V.C of the paper, evaluated once in fp64 and frozen into integer tables.
int build_tables(nhp_planner *p)
{
    const int n = p->n, nt = p->nt;
    p->beta.resize(nt); p->psi2.resize(nt); p->I.resize(nt); p->J.resize(nt);
    p->B.resize((size_t)nt * n); p->len_q.resize((size_t)6 * nt); p->cosq.resize(nt); p->sinq.resize(nt);
    const double one = (double)(1u << p->w.cost_one_log2);
    for (int t = 0; t < nt; t++) {
        const double s = sin_frac(t, nt), c = sin_frac(t + nt / 4, nt);
        // alpha = R sin(theta); zeta(x) = round(2x)/2; beta = floor(zeta(alpha)); Psi = zeta - beta  (l.233-240)
        const double z = std::round(2.0 * (p->R * s)) / 2.0;
        const double fl = std::floor(z);
        p->beta[t] = (int32_t)fl;
        p->psi2[t] = (uint8_t)(int)(2.0 * (z - fl));
        // eq (19) on the integer octant; eq (20); eq (24)
        const int o = t & (nt / 2 - 1);
        const int I = (o <= nt / 8 || o >= 3 * nt / 8) ? 0 : 1;
        const double K = I == 0 ? s / c : c / s, f = I == 0 ? c : s;
        p->I[t] = (uint8_t)I;
        p->J[t] = (int8_t)(f > 0 ? 1 : -1);
        for (int y = 0; y < n; y++) p->B[(size_t)t * n + y] = (int32_t)std::round((double)y * K);   // l.284
        // edge lengths l.334 -> fixed point
        const double lt = 2.0 * kPi * p->R / (double)nt, ls = 1.0 / std::fabs(f);
        for (int m = 0; m < 6; m++) {
            const double len = (m == M_SF || m == M_SB) ? ls : lt;
            const double q = std::round(one * len * (double)p->w.dir_mult[m] / 256.0);
            if (q < 1.0 || q * 255.0 / 16.0 >= (double)(1u << 26)) return NHP_E_WEIGHTS;
            p->len_q[(size_t)m * nt + t] = (uint32_t)q;
        }
        p->cosq[t] = (int32_t)std::round(16384.0 * c);
        p->sinq[t] = (int32_t)std::round(16384.0 * s);
    }
    for (int m = 0; m < 6; m++)
        if (p->w.ct[m] >= (1u << 26)) return NHP_E_WEIGHTS;
    return NHP_OK;
}

int upload_tables(nhp_planner *p)
{
    const int n = p->n, nt = p->nt;
    std::vector<int16_t> beta16(nt), B16((size_t)nt * n);
    std::vector<uint8_t> IJ(nt);
    std::vector<int32_t> rot((size_t)4 * nt);
    for (int t = 0; t < nt; t++) {
        beta16[t] = (int16_t)p->beta[t];
        IJ[t] = (uint8_t)(p->I[t] | ((p->J[t] > 0 ? 1 : 0) << 1));
        rot[4 * t + 0] = p->cosq[t]; rot[4 * t + 1] = p->sinq[t];
        rot[4 * t + 2] = p->psi2[t]; rot[4 * t + 3] = p->psi2[(t + nt / 4) & (nt - 1)];   // 2 Psi0, 2 Psi1, eq (16)
    }
    for (size_t k = 0; k < B16.size(); k++) B16[k] = (int16_t)p->B[k];
    std::vector<int16_t> tlist;
    for (int t = 0; t < nt; t++) if (p->I[t] == 0) tlist.push_back((int16_t)t);
    p->n_xslices = (int)tlist.size();
    for (int t = 0; t < nt; t++) if (p->I[t] != 0) tlist.push_back((int16_t)t);
    CU(cudaMalloc(&p->d_tlist, sizeof(int16_t) * nt));
    CU(cudaMemcpyAsync(p->d_tlist, tlist.data(), sizeof(int16_t) * nt, cudaMemcpyHostToDevice, p->stream));
    CU(cudaMalloc(&p->d_beta, sizeof(int16_t) * nt));
    CU(cudaMalloc(&p->d_B, sizeof(int16_t) * B16.size()));
    CU(cudaMalloc(&p->d_lenq, sizeof(uint32_t) * 6 * nt));
    CU(cudaMalloc(&p->d_IJ, nt));
    CU(cudaMalloc(&p->d_rot, sizeof(int32_t) * 4 * nt));
    CU(cudaMemcpyAsync(p->d_beta, beta16.data(), sizeof(int16_t) * nt, cudaMemcpyHostToDevice, p->stream));
    CU(cudaMemcpyAsync(p->d_B, B16.data(), sizeof(int16_t) * B16.size(), cudaMemcpyHostToDevice, p->stream));
    CU(cudaMemcpyAsync(p->d_lenq, p->len_q.data(), sizeof(uint32_t) * 6 * nt, cudaMemcpyHostToDevice, p->stream));
    CU(cudaMemcpyAsync(p->d_IJ, IJ.data(), nt, cudaMemcpyHostToDevice, p->stream));
    CU(cudaMemcpyAsync(p->d_rot, rot.data(), sizeof(int32_t) * 4 * nt, cudaMemcpyHostToDevice, p->stream));
    // x-rows kernel (straight.cu: straight_xl_kernel): what tile T (columns 32 T .. 32 T + 31) of an I = 0 slice needs that depends
    // only on (slice, T).  delta_k = B(32 T + k) - bmin is the row of line 0 at column k relative to the tile's first row; the
    // 8-column sector group m = k / 8 is fetched sheared by dlo8(m) = its smallest delta.  Word of lane k:
    //     dq_k = delta_k - dlo8(m)  (bits 0-2)  |  rows the group needs = 32 + max dq  (bits 8-13)  |  bmin + dlo8(m)  (bits 16-31, signed)
    std::vector<uint32_t> xl;
    if (n >= 32) {
        const int NT = n / 32, nx = p->n_xslices;
        xl.assign((size_t)nx * NT * 32, 0u);
        for (int xs = 0; xs < nx; xs++) {
            const int32_t *Bt = p->B.data() + (size_t)tlist[xs] * n;
            for (int T = 0; T < NT; T++) {
                int bmin = 1 << 30;
                for (int k = 0; k < 32; k++) bmin = Bt[32 * T + k] < bmin ? Bt[32 * T + k] : bmin;
                for (int m8 = 0; m8 < 4; m8++) {
                    int lo = 1 << 30, hi = -(1 << 30);
                    for (int e = 0; e < 8; e++) { const int d = Bt[32 * T + 8 * m8 + e] - bmin; lo = d < lo ? d : lo; hi = d > hi ? d : hi; }
                    if (hi - lo > 7 || bmin + lo < -32768 || bmin + lo > 32767) return fail(p, NHP_E_ARG, "x-rows table: slope of a straight line exceeds 1");
                    for (int e = 0; e < 8; e++) {
                        const int k = 8 * m8 + e, dq = Bt[32 * T + k] - bmin - lo;
                        xl[((size_t)xs * NT + T) * 32 + k] = (uint32_t)dq | ((uint32_t)(32 + hi - lo) << 8) | ((uint32_t)(bmin + lo) << 16);
                    }
                }
            }
        }
        CU(cudaMalloc(&p->d_xl_tab, sizeof(uint32_t) * xl.size() + 16));
        CU(cudaMemcpyAsync(p->d_xl_tab, xl.data(), sizeof(uint32_t) * xl.size(), cudaMemcpyHostToDevice, p->stream));
    }
    CU(cudaStreamSynchronize(p->stream));            // the staging vectors die with this scope
    return NHP_OK;
}

bool in_grid(const nhp_planner *p, int i, int j, int t) { return i >= 0 && j >= 0 && t >= 0 && i < p->n && j < p->n && t < p->nt; }

// Everything that scales with the grid or the limits lives in the caller's workspace (no allocation during
// processing).  Offsets in bytes, each 256-byte aligned.
struct WsLayout {
    nhp_limits lim;                 // resolved
    int side, sidew, cap_levels;
    size_t cap_runs;
    size_t soft_copies, reach, mask, E, runs, run_off, Hk, Mk, total;
};

WsLayout workspace_layout(int log2_n, int log2_nt, int flags, const nhp_limits *lim)
{
    WsLayout L{};
    const size_t n = (size_t)1 << log2_n, nt = (size_t)1 << log2_nt, nr = n * n * nt;
    int rmax = (lim && lim->max_footprint_radius > 0) ? lim->max_footprint_radius : 64;
    if (rmax > (int)n / 2 - 1) rmax = (int)n / 2 - 1;
    L.lim.max_footprint_radius = rmax;
    L.lim.max_reach_levels = (lim && lim->max_reach_levels > 0) ? lim->max_reach_levels : 0;
    L.side = 2 * rmax + 1; L.sidew = (L.side + 31) / 32;
    L.cap_levels = 1;
    while ((2 << (L.cap_levels - 1)) <= L.side) L.cap_levels++;            // floor(log2 side) + 1 levels of the sparse tables
    L.cap_runs = nt * (size_t)L.side * 4 + 1;                              // <= 4 runs per footprint row on average
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
    L.soft_copies = take((flags & NHP_FLAG_SOFT) ? 3 * nr : 0);            // S_left, S_right, S_line
    L.reach = take(L.lim.max_reach_levels > 0 ? ((size_t)L.lim.max_reach_levels + 4) * (nr / 8) : 0);
    L.mask = take((size_t)L.side * L.side);
    L.E = take(sizeof(uint32_t) * nt * L.side * L.sidew);
    L.runs = take(sizeof(int4) * L.cap_runs);
    L.run_off = take(sizeof(int32_t) * (nt + 1));
    L.Hk = take((n * n / 8) * L.cap_levels);
    L.Mk = take((flags & NHP_FLAG_SOFT) ? n * n * L.cap_levels : 0);
    L.total = off;
    return L;
}

// Status words and the first NHP_PLAN_EAGER waypoints come back in one copy (they are contiguous on the device); the rest
// of a longer plan, rarely, in a second one.  Step 8.
int fetch_plan(nhp_planner *p, const int32_t *d_st)
{
    const size_t head = sizeof(int32_t) * NHP_STATUS_WORDS;
    CU(cudaMemcpyAsync(p->h_status, d_st, head + sizeof(nhp_waypoint) * p->plan_eager, cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    const int n = p->h_status[2];
    if (p->h_status[1] == NHP_OK && n > p->plan_eager) {
        const size_t done = head + sizeof(nhp_waypoint) * p->plan_eager;
        CU(cudaMemcpyAsync((uint8_t *)p->h_status + done, (const uint8_t *)d_st + done, sizeof(nhp_waypoint) * (size_t)(n - p->plan_eager),
                           cudaMemcpyDeviceToHost, p->stream));
        CU(cudaStreamSynchronize(p->stream));
    }
    return NHP_OK;
}

}  // namespace

bool prof_grow(nhp_planner *p)
{
    const size_t pairs = p->ev.size() / 2;
    if (pairs + PROF_GROW > (size_t)PROF_MAX_PAIRS) return false;
    std::vector<cudaEvent_t> more(2 * PROF_GROW, nullptr);
    for (auto &e : more)
        if (cudaEventCreate(&e) != cudaSuccess) {
            for (auto &f : more) if (f) cudaEventDestroy(f);
            return false;
        }
    p->ev.insert(p->ev.end(), more.begin(), more.end());
    p->ev_slot.resize(pairs + PROF_GROW, 0);
    return true;
}

extern "C" {

int nhp_query_sizes(int log2_n, int log2_ntheta, int flags, const nhp_limits *lim, nhp_sizes *out)
{
    if (!out) return NHP_E_ARG;
    if (log2_n < 5 || log2_n > 12 || log2_ntheta < 5 || log2_ntheta > 12) return NHP_E_NOT_POW2;
    if (lim && (lim->max_footprint_radius < 0 || lim->max_reach_levels < 0 || lim->max_reach_levels > 254)) return NHP_E_ARG;
    const size_t nr = ((size_t)1 << (2 * log2_n)) << log2_ntheta;
    out->V_bytes = nr * 4;
    out->C_bytes = nr / 8;
    out->S_bytes = (flags & NHP_FLAG_SOFT) ? nr : 0;
    out->workspace_bytes = workspace_layout(log2_n, log2_ntheta, flags, lim).total;
    return NHP_OK;
}

int nhp_planner_create(nhp_planner **out, int log2_n, int log2_ntheta, double R_cells, const nhp_weights *w,
                       const nhp_limits *lim, const nhp_buffers *dev, void *cuda_stream)
{
    if (!out || !w || !dev) return NHP_E_ARG;
    *out = nullptr;
    if (log2_n < 5 || log2_n > 12 || log2_ntheta < 5 || log2_ntheta > 12) return NHP_E_NOT_POW2;
    if (!(R_cells >= 1.0) || w->cost_one_log2 < 0 || w->cost_one_log2 > 16) return NHP_E_ARG;
    if (lim && (lim->max_footprint_radius < 0 || lim->max_reach_levels < 0 || lim->max_reach_levels > 254)) return NHP_E_ARG;
    if ((double)(1 << log2_ntheta) < 2.0 * kPi * R_cells) return NHP_E_ANGRES;
    if (!dev->V || !dev->C || !dev->workspace || ((w->flags & NHP_FLAG_SOFT) && !dev->S)) return NHP_E_BUFFER;
    if (((uintptr_t)dev->V | (uintptr_t)dev->C | (uintptr_t)dev->S | (uintptr_t)dev->workspace) & 255) return NHP_E_BUFFER;
    nhp_planner *p = new (std::nothrow) nhp_planner();
    if (!p) return NHP_E_ARG;
    p->log2_n = log2_n; p->log2_nt = log2_ntheta; p->n = 1 << log2_n; p->nt = 1 << log2_ntheta;
    p->R = R_cells; p->w = *w; p->stream = (cudaStream_t)cuda_stream;
    p->V = (uint32_t *)dev->V; p->C = (uint32_t *)dev->C; p->S = (w->flags & NHP_FLAG_SOFT) ? (uint8_t *)dev->S : nullptr;
    // the device that owns the caller's buffers is the handle's device
    cudaPointerAttributes attr{};
    if (cudaPointerGetAttributes(&attr, dev->V) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        delete p;
        return NHP_E_BUFFER;
    }
    p->device = attr.device;
    for (const void *b : {(const void *)dev->C, (const void *)p->S, (const void *)dev->workspace}) {       // one device owns them all
        cudaPointerAttributes a{};
        if (b && (cudaPointerGetAttributes(&a, b) != cudaSuccess || a.type != cudaMemoryTypeDevice || a.device != p->device)) {
            cudaGetLastError();
            delete p;
            return NHP_E_BUFFER;
        }
    }
    DeviceGuard guard(p);
    // carve the workspace
    const WsLayout L = workspace_layout(log2_n, log2_ntheta, w->flags, lim);
    p->lim = L.lim;
    uint8_t *ws = (uint8_t *)dev->workspace;
    const size_t nr = (size_t)p->n * p->n * p->nt;
    if (p->S) { p->S_left = ws + L.soft_copies; p->S_right = p->S_left + nr; p->S_line = p->S_right + nr; }
    if (L.lim.max_reach_levels > 0) {
        const size_t W = nr / 32;
        p->r_Lt = (uint32_t *)(ws + L.reach); p->r_Ct = p->r_Lt + W; p->r_Gt = p->r_Ct + W; p->r_levels = p->r_Gt + W;
    }
    p->d_mask = ws + L.mask; p->d_E = (uint32_t *)(ws + L.E);
    p->d_runs = (int4 *)(ws + L.runs); p->d_run_off = (int32_t *)(ws + L.run_off);
    p->d_Hk = (uint32_t *)(ws + L.Hk); p->d_Mk = p->S ? ws + L.Mk : nullptr;
    p->cap_runs = L.cap_runs; p->cap_levels = L.cap_levels;
    int rc = build_tables(p);
    if (rc == NHP_OK) rc = upload_tables(p);
    const size_t npx = (size_t)p->n * p->n;
    p->plan_cap = NHP_PLAN_CAP;
    const size_t sp_bytes = sizeof(int32_t) * NHP_STATUS_WORDS + sizeof(nhp_waypoint) * p->plan_cap;      // status words + plan
    auto alloc = [&](void **ptr, size_t bytes) { if (rc == NHP_OK && cudaMalloc(ptr, bytes) != cudaSuccess) rc = NHP_E_CUDA; };
    alloc((void **)&p->d_hard, npx);
    alloc((void **)&p->d_soft, npx);
    if (w->flags & NHP_FLAG_SOFT) alloc((void **)&p->d_dtg, sizeof(int32_t) * npx);
    if (w->flags & NHP_FLAG_SOFT) { alloc((void **)&p->d_lane_dir, npx); alloc((void **)&p->d_lane_pen, npx); }
    alloc((void **)&p->d_status, 2 * sp_bytes);
    alloc((void **)&p->d_goals, sizeof(int32_t) * 3 * NHP_MAX_GOALS);
    if (rc == NHP_OK && cudaMallocHost((void **)&p->h_status, sp_bytes) != cudaSuccess) rc = NHP_E_CUDA;
    if (rc == NHP_OK) {
        p->d_plan = (nhp_waypoint *)(p->d_status + NHP_STATUS_WORDS);
        p->d_rstatus = (int32_t *)((uint8_t *)p->d_status + sp_bytes);
        p->d_rplan = (nhp_waypoint *)(p->d_rstatus + NHP_STATUS_WORDS);
        p->h_plan = (nhp_waypoint *)(p->h_status + NHP_STATUS_WORDS);
        if (cudaMemsetAsync(p->d_status, 0, 2 * sp_bytes, p->stream) != cudaSuccess) rc = NHP_E_CUDA;
    }
    if (rc == NHP_OK) rc = set_kernel_attributes(p);
    if (rc == NHP_OK) rc = build_cycle_graph(p);
    if (rc != NHP_OK) { nhp_planner_destroy(p); return rc; }
    *out = p;
    return NHP_OK;
}

int nhp_planner_destroy(nhp_planner *p)
{
    if (!p) return NHP_E_ARG;
    {
        DeviceGuard guard(p);
        cudaStreamSynchronize(p->stream);
        if (p->cycle_exec) cudaGraphExecDestroy(p->cycle_exec);
        if (p->cycle_graph) cudaGraphDestroy(p->cycle_graph);
        cudaFree(p->d_beta); cudaFree(p->d_B); cudaFree(p->d_lenq); cudaFree(p->d_IJ); cudaFree(p->d_rot); cudaFree(p->d_tlist); cudaFree(p->d_xl_tab);
        cudaFree(p->d_hard); cudaFree(p->d_soft); cudaFree(p->d_status); cudaFree(p->d_dtg); cudaFree(p->d_goals);
        cudaFree(p->d_lane_dir); cudaFree(p->d_lane_pen);
        if (p->h_status) cudaFreeHost(p->h_status);
        for (auto &e : p->ev) if (e) cudaEventDestroy(e);
    }
    delete p;
    return NHP_OK;
}

const char *nhp_last_error(const nhp_planner *p) { return p ? p->err.c_str() : "null handle"; }

int nhp_render_vehicle_footprint(nhp_planner *p, const uint8_t *mask_host, int mw, int mh, double origin_u, double origin_v)
{
    if (!p || !mask_host || mw < 1 || mh < 1 || mw > 1024 || mh > 1024) return fail(p, NHP_E_ARG, "bad footprint mask");
    // circumscribed radius of the mask around the vehicle origin, in cells (+2 for Psi and rounding)
    const double mu = std::fmax(std::fabs(-origin_u - 0.5), std::fabs((double)mw - 1.0 - origin_u + 0.5));
    const double mv = std::fmax(std::fabs(-origin_v - 0.5), std::fabs((double)mh - 1.0 - origin_v + 0.5));
    const int rad = (int)std::ceil(std::hypot(mu, mv)) + 2;
    if (2 * rad >= p->n) return fail(p, NHP_E_ARG, "footprint does not fit the grid");
    if (rad > p->lim.max_footprint_radius) return fail(p, NHP_E_BUFFER, "footprint radius exceeds nhp_limits.max_footprint_radius");
    DeviceGuard guard(p);
    p->have_footprint = false;
    p->rad = rad; p->side = 2 * rad + 1; p->sidew = (p->side + 31) / 32;
    CU(cudaMemcpyAsync(p->d_mask, mask_host, (size_t)mw * mh, cudaMemcpyHostToDevice, p->stream));
    const int64_t ouq = (int64_t)std::llround(origin_u * 32768.0), ovq = (int64_t)std::llround(origin_v * 32768.0);
    p->launches += launch_footprint_raster(p, mw, mh, ouq, ovq);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(p->stream));            // mask_host may be freed by the caller after return
    const int frc = finish_footprint(p);
    if (frc != NHP_OK) return fail(p, frc, frc == NHP_E_BUFFER ? "footprint mask breaks into more runs than the workspace holds" : "building the footprint run tables failed");
    p->have_footprint = true;
    p->have_render = false;
    p->have_run = false;
    p->r_n_levels = -1;
    return NHP_OK;
}

int nhp_set_box(nhp_planner *p, int f, int r, int s)
{
    if (!p || f < 0 || r < 0 || s < 1 || f + r < 1 || f + r > 1024 || 2 * s > 1024) return fail(p, NHP_E_ARG, "bad bounding box");
    // vehicle-frame rectangle u in [-r, f), v in [-s, s): all-ones mask, pixel 0 centred at (-r + 1/2, -s + 1/2)
    const std::vector<uint8_t> mask((size_t)(f + r) * (2 * s), 1);
    return nhp_render_vehicle_footprint(p, mask.data(), f + r, 2 * s, (double)r - 0.5, (double)s - 0.5);
}

int nhp_render_obstacles(nhp_planner *p, const uint8_t *hard, const uint8_t *soft, int on_device)
{
    if (!p || !hard) return fail(p, NHP_E_ARG, "hard image is NULL");
    if (!p->have_footprint) return fail(p, NHP_E_STATE, "render_obstacles before render_vehicle_footprint");
    const bool want_soft = p->S != nullptr;
    if (want_soft && !soft) return fail(p, NHP_E_ARG, "NHP_FLAG_SOFT planner needs a soft image");
    if (!want_soft && soft) return fail(p, NHP_E_ARG, "soft image given but the planner has no soft volume");
    DeviceGuard guard(p);
    const size_t npx = (size_t)p->n * p->n;
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CU(cudaMemcpyAsync(p->d_hard, hard, npx, kind, p->stream));                       // step 3
    if (want_soft) CU(cudaMemcpyAsync(p->d_soft, soft, npx, kind, p->stream));
    p->launches += launch_render(p, want_soft);                                       // step 4
    CU(cudaGetLastError());
    p->have_render = true;
    p->have_run = false;                  // both planners' results belong to the previous collision volume
    p->r_n_levels = -1;
    return NHP_OK;
}

int nhp_set_lane_penalty(nhp_planner *p, const uint8_t *lane_dir, const uint8_t *lane_pen, int on_device)
{
    if (!p) return NHP_E_ARG;
    if (!p->S || !p->d_lane_dir) return fail(p, NHP_E_ARG, "the planner has no soft volume (NHP_FLAG_SOFT)");
    if (!lane_dir != !lane_pen) return fail(p, NHP_E_ARG, "lane_dir and lane_pen must both be given or both be NULL");
    if (!lane_dir) { p->have_lane = false; return NHP_OK; }
    DeviceGuard guard(p);
    const size_t npx = (size_t)p->n * p->n;
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CU(cudaMemcpyAsync(p->d_lane_dir, lane_dir, npx, kind, p->stream));
    CU(cudaMemcpyAsync(p->d_lane_pen, lane_pen, npx, kind, p->stream));
    p->have_lane = true;
    return NHP_OK;
}

int nhp_render_obstacles_dt(nhp_planner *p, const uint8_t *hard, int on_device, double k, float *dist_dev_out)
{
    if (!p || !hard) return fail(p, NHP_E_ARG, "hard image is NULL");
    if (!(k >= 0.0) || k > 64.0) return fail(p, NHP_E_ARG, "k outside [0, 64]");
    if (!p->have_footprint) return fail(p, NHP_E_STATE, "render_obstacles before render_vehicle_footprint");
    if (!p->S || !p->d_dtg) return fail(p, NHP_E_ARG, "the planner has no soft volume (NHP_FLAG_SOFT)");
    DeviceGuard guard(p);
    const size_t npx = (size_t)p->n * p->n;
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CU(cudaMemcpyAsync(p->d_hard, hard, npx, kind, p->stream));
    p->launches += launch_soft_from_hard(p, (float)k, dist_dev_out, nullptr);        // steps 1-2
    p->launches += launch_render(p, true);                                            // step 4
    CU(cudaGetLastError());
    p->have_render = true;
    p->have_run = false;
    p->r_n_levels = -1;
    return NHP_OK;
}

int nhp_debug_cycle_graph_kernels(const nhp_planner *p)
{
    return (p && p->cycle_exec) ? p->cycle_graph_kernels : 0;
}

int nhp_debug_set_plan_eager(nhp_planner *p, int n_waypoints)
{
    if (!p) return NHP_E_ARG;
    if (n_waypoints < 1 || n_waypoints > NHP_PLAN_CAP) return fail(p, NHP_E_ARG, "n_waypoints outside [1, plan capacity]");
    p->plan_eager = n_waypoints;
    return NHP_OK;
}

int nhp_debug_soft_image(nhp_planner *p, uint8_t *soft_host)
{
    if (!p || !soft_host) return fail(p, NHP_E_ARG, "NULL argument");
    if (!p->S || !p->have_render) return fail(p, NHP_E_STATE, "no soft image rendered yet");
    DeviceGuard guard(p);
    CU(cudaMemcpyAsync(soft_host, p->d_soft, (size_t)p->n * p->n, cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    return NHP_OK;
}

int nhp_run_nturn(nhp_planner *p, int i, int j, int theta, int n_cycles)
{
    return nhp_run_nturn_from(p, i, j, theta, -1, n_cycles);
}

int nhp_run_nturn_from(nhp_planner *p, int i, int j, int theta, int m0, int n_cycles)
{
    if (!p) return NHP_E_ARG;
    if (m0 < -1 || m0 > 5) return fail(p, NHP_E_ARG, "maneuver id outside [-1, 5]");
    if (m0 >= 0 && (p->w.flags & NHP_FLAG_FORWARD_ONLY) && (m0 == M_RB || m0 == M_SB || m0 == M_LB))
        return fail(p, NHP_E_ARG, "a reverse maneuver cannot be in progress with NHP_FLAG_FORWARD_ONLY");
    if (!p->have_render) return fail(p, NHP_E_STATE, "run_nturn before render_obstacles");
    if (!in_grid(p, i, j, theta)) return fail(p, NHP_E_ARG, "start pose outside the grid");
    if (n_cycles <= 0) n_cycles = NHP_DEFAULT_CYCLES;
    DeviceGuard guard(p);
    p->start[0] = i; p->start[1] = j; p->start[2] = theta;
    p->start_m0 = m0;
    p->launches += launch_init_volume(p, i, j, theta);
    p->canonical = false;
    if (m0 >= 0) p->launches += launch_seed_in_progress(p, m0);
    p->launches += launch_cycles(p, n_cycles, true);
    CU(cudaGetLastError());
    p->have_run = true;
    return NHP_OK;
}

int nhp_reach_run(nhp_planner *p, int i, int j, int theta, int n_levels)
{
    if (!p) return NHP_E_ARG;
    if (!p->have_render) return fail(p, NHP_E_STATE, "reach_run before render_obstacles");
    if (!in_grid(p, i, j, theta)) return fail(p, NHP_E_ARG, "start pose outside the grid");
    if (n_levels <= 0) n_levels = NHP_DEFAULT_CYCLES;
    if (n_levels > 254) return fail(p, NHP_E_ARG, "more than 254 levels");
    if (n_levels > p->lim.max_reach_levels) return fail(p, NHP_E_BUFFER, "n_levels exceeds nhp_limits.max_reach_levels of this planner");
    DeviceGuard guard(p);
    int k = 0;
    const int rc = launch_reach_run(p, i, j, theta, n_levels, &k);
    if (rc != NHP_OK) return fail(p, rc, "launching the level sweeps failed");
    p->launches += k;
    p->r_start[0] = i; p->r_start[1] = j; p->r_start[2] = theta;
    CU(cudaGetLastError());
    return NHP_OK;
}

int nhp_reach_levels(nhp_planner *p, const uint32_t **dev_ptr_out, int *n_levels)
{
    if (!p || !dev_ptr_out || !n_levels) return fail(p, NHP_E_ARG, "NULL argument");
    if (p->r_n_levels < 0) return fail(p, NHP_E_STATE, "reach_levels before reach_run");
    *dev_ptr_out = p->r_levels;
    *n_levels = p->r_n_levels;
    return NHP_OK;
}

int nhp_reach_count_volume(nhp_planner *p, uint8_t *K_dev)
{
    if (!p || !K_dev) return fail(p, NHP_E_ARG, "NULL argument");
    if (p->r_n_levels < 0) return fail(p, NHP_E_STATE, "reach_count_volume before reach_run");
    if ((uintptr_t)K_dev & 15) return fail(p, NHP_E_BUFFER, "K buffer must be 16-byte aligned");
    DeviceGuard guard(p);
    p->launches += launch_reach_count(p, K_dev);
    CU(cudaGetLastError());
    return NHP_OK;
}

int nhp_reach_extract_path(nhp_planner *p, int gi, int gj, int gtheta, nhp_waypoint *out_host, int cap, int *count, int *n_maneuvers)
{
    if (!p || !out_host || !count || !n_maneuvers || cap < 1) return fail(p, NHP_E_ARG, "bad reach_extract_path argument");
    if (p->r_n_levels < 0) return fail(p, NHP_E_STATE, "reach_extract_path before reach_run");
    if (!in_grid(p, gi, gj, gtheta)) return fail(p, NHP_E_ARG, "goal pose outside the grid");
    *count = 0; *n_maneuvers = -1;
    DeviceGuard guard(p);
    p->launches += launch_reach_backtrack(p, gi, gj, gtheta);
    CU(cudaGetLastError());
    if (fetch_plan(p, p->d_rstatus) != NHP_OK) return NHP_E_CUDA;
    const int rc = p->h_status[1];
    if (rc == NHP_E_START_BLOCKED) return fail(p, rc, "the start vertex collides");
    if (rc == NHP_E_GOAL_UNREACHED) return fail(p, rc, "goal not reached within the levels of the last reach_run");
    if (rc != NHP_OK) return fail(p, rc, "plan longer than the internal buffer");
    const int n = p->h_status[2];
    if (n > cap) return fail(p, NHP_E_BUFFER, "plan longer than the caller's buffer");
    std::memcpy(out_host, p->h_plan, sizeof(nhp_waypoint) * n);
    *count = n;
    *n_maneuvers = p->h_status[3];
    return NHP_OK;
}

int nhp_run_more(nhp_planner *p, int n_cycles)
{
    if (!p) return NHP_E_ARG;
    if (!p->have_run) return fail(p, NHP_E_STATE, "run_more before run_nturn");
    if (n_cycles <= 0) return fail(p, NHP_E_ARG, "n_cycles must be positive");
    DeviceGuard guard(p);
    if (p->canonical) { p->launches += launch_export_volume(p, false); p->canonical = false; }
    p->launches += launch_cycles(p, n_cycles, false);
    CU(cudaGetLastError());
    return NHP_OK;
}

int nhp_cost_volume(nhp_planner *p, const uint32_t **dev_ptr_out)
{
    if (!p || !dev_ptr_out) return NHP_E_ARG;
    if (!p->have_run) return fail(p, NHP_E_STATE, "cost_volume before run_nturn");
    DeviceGuard guard(p);
    if (!p->canonical) { p->launches += launch_export_volume(p, true); p->canonical = true; }
    CU(cudaGetLastError());
    *dev_ptr_out = p->V;
    return NHP_OK;
}

int nhp_status(nhp_planner *p)
{
    if (!p) return NHP_E_ARG;
    DeviceGuard guard(p);
    CU(cudaMemcpyAsync(p->h_status, p->d_status, sizeof(int32_t) * NHP_STATUS_WORDS, cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    if (p->have_run && p->h_status[0]) return fail(p, NHP_E_START_BLOCKED, "the start vertex collides");
    return NHP_OK;
}

int nhp_extract_path(nhp_planner *p, int gi, int gj, int gtheta, nhp_waypoint *out_host, int cap, int *count, uint32_t *cost)
{
    if (!p || !out_host || !count || !cost || cap < 1) return fail(p, NHP_E_ARG, "bad extract_path argument");
    if (!p->have_run) return fail(p, NHP_E_STATE, "extract_path before run_nturn");
    if (!in_grid(p, gi, gj, gtheta)) return fail(p, NHP_E_ARG, "goal pose outside the grid");
    *count = 0; *cost = NHP_INF;
    DeviceGuard guard(p);
    if (p->canonical) { p->launches += launch_export_volume(p, false); p->canonical = false; }
    p->launches += launch_backtrack(p, gi, gj, gtheta);
    CU(cudaGetLastError());
    if (fetch_plan(p, p->d_status) != NHP_OK) return NHP_E_CUDA;                      // step 8
    const int rc = p->h_status[1];
    if (rc == NHP_E_START_BLOCKED) return fail(p, rc, "the start vertex collides");
    if (rc == NHP_E_GOAL_UNREACHED) return fail(p, rc, "goal not reached");
    if (rc != NHP_OK) return fail(p, rc, "plan longer than the internal buffer");
    const int n = p->h_status[2];
    if (n > cap) return fail(p, NHP_E_BUFFER, "plan longer than the caller's buffer");
    std::memcpy(out_host, p->h_plan, sizeof(nhp_waypoint) * n);
    *count = n;
    *cost = (uint32_t)p->h_status[3];
    return NHP_OK;
}

int nhp_extract_path_goalset(nhp_planner *p, const int32_t *goals_host, int n_goals, int d, uint32_t W, uint32_t w,
                             nhp_waypoint *out_host, int cap, int *count, uint32_t *cost, int32_t *chosen, uint64_t *score)
{
    if (!p || !goals_host || !out_host || !count || !cost || cap < 1) return fail(p, NHP_E_ARG, "bad extract_path_goalset argument");
    if (n_goals < 1 || n_goals > NHP_MAX_GOALS || d < 0 || d > 31 || W >= (1u << 20) || w >= (1u << 20))
        return fail(p, NHP_E_ARG, "goal set outside the supported range (<= 256 goals, d <= 31, W, w < 2^20)");
    if ((long long)n_goals * (2 * d + 1) * (2 * d + 1) * (2 * d + 1) >= (1ll << 24)) return fail(p, NHP_E_ARG, "goal set too large");
    if (!p->have_run) return fail(p, NHP_E_STATE, "extract_path before run_nturn");
    for (int g = 0; g < n_goals; g++)
        if (!in_grid(p, goals_host[3 * g], goals_host[3 * g + 1], goals_host[3 * g + 2])) return fail(p, NHP_E_ARG, "goal pose outside the grid");
    *count = 0; *cost = NHP_INF;
    DeviceGuard guard(p);
    if (p->canonical) { p->launches += launch_export_volume(p, false); p->canonical = false; }
    CU(cudaMemcpyAsync(p->d_goals, goals_host, sizeof(int32_t) * 3 * n_goals, cudaMemcpyHostToDevice, p->stream));
    p->launches += launch_goal_search(p, n_goals, d, W, w);                           // step 6
    p->launches += launch_backtrack(p, -1, -1, -1);                                   // step 7
    CU(cudaGetLastError());
    if (fetch_plan(p, p->d_status) != NHP_OK) return NHP_E_CUDA;                      // step 8
    const int rc = p->h_status[1];
    if (rc == NHP_E_START_BLOCKED) return fail(p, rc, "the start vertex collides");
    if (rc == NHP_E_GOAL_UNREACHED) return fail(p, rc, "no vertex of the goal set is reached");
    if (rc != NHP_OK) return fail(p, rc, "plan longer than the internal buffer");
    const int n = p->h_status[2];
    if (n > cap) return fail(p, NHP_E_BUFFER, "plan longer than the caller's buffer");
    std::memcpy(out_host, p->h_plan, sizeof(nhp_waypoint) * n);
    *count = n;
    *cost = (uint32_t)p->h_status[3];
    if (chosen) for (int k = 0; k < 4; k++) chosen[k] = p->h_status[4 + k];
    if (score) *score = (uint64_t)(uint32_t)p->h_status[8] | ((uint64_t)(uint32_t)p->h_status[9] << 32);
    return NHP_OK;
}

int nhp_index_to_pose(const nhp_planner *p, int i, int j, int theta, double *x, double *y, double *theta_rad)
{
    if (!p || !x || !y || !theta_rad || !in_grid(p, i, j, theta)) return NHP_E_ARG;
    *x = i + p->psi2[theta] / 2.0;                                                    // eq (16)
    *y = j + p->psi2[(theta + p->nt / 4) & (p->nt - 1)] / 2.0;
    *theta_rad = 2.0 * kPi * theta / p->nt;
    return NHP_OK;
}

int nhp_pose_to_index(const nhp_planner *p, double x, double y, double theta_rad, int *i, int *j, int *theta)
{
    if (!p || !i || !j || !theta) return NHP_E_ARG;
    const int t = (int)std::llround(theta_rad / (2.0 * kPi) * p->nt) & (p->nt - 1);
    const long long ii = std::llround(x - p->psi2[t] / 2.0), jj = std::llround(y - p->psi2[(t + p->nt / 4) & (p->nt - 1)] / 2.0);
    if (ii < 0 || jj < 0 || ii >= p->n || jj >= p->n) return NHP_E_ARG;
    *i = (int)ii; *j = (int)jj; *theta = t;
    return NHP_OK;
}

int nhp_debug_tables(const nhp_planner *p, int32_t *beta, uint8_t *psi2, int32_t *B, uint8_t *I, int8_t *J, uint32_t *len_q)
{
    if (!p) return NHP_E_ARG;
    if (beta) std::memcpy(beta, p->beta.data(), sizeof(int32_t) * p->nt);
    if (psi2) std::memcpy(psi2, p->psi2.data(), p->nt);
    if (B) std::memcpy(B, p->B.data(), sizeof(int32_t) * p->B.size());
    if (I) std::memcpy(I, p->I.data(), p->nt);
    if (J) std::memcpy(J, p->J.data(), p->nt);
    if (len_q) std::memcpy(len_q, p->len_q.data(), sizeof(uint32_t) * p->len_q.size());
    return NHP_OK;
}

long long nhp_launch_count(const nhp_planner *p) { return p ? p->launches : 0; }

long long nhp_prof_dropped(const nhp_planner *p) { return p ? p->ev_dropped : 0; }

int nhp_debug_footprint(nhp_planner *p, int *radius, uint8_t *covered, size_t cap)
{
    if (!p || !radius) return fail(p, NHP_E_ARG, "NULL argument");
    if (!p->have_footprint) return fail(p, NHP_E_STATE, "no footprint rendered yet");
    *radius = p->rad;
    if (!covered) return NHP_OK;
    const size_t side = (size_t)p->side, need = (size_t)p->nt * side * side;
    if (cap < need) return fail(p, NHP_E_BUFFER, "covered[] too small");
    DeviceGuard guard(p);
    std::vector<uint32_t> E((size_t)p->nt * side * p->sidew);
    CU(cudaMemcpyAsync(E.data(), p->d_E, sizeof(uint32_t) * E.size(), cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    for (size_t t = 0; t < (size_t)p->nt; t++)
        for (size_t r = 0; r < side; r++)
            for (size_t c = 0; c < side; c++)
                covered[(t * side + r) * side + c] = (E[(t * side + r) * p->sidew + (c >> 5)] >> (c & 31)) & 1u;
    return NHP_OK;
}

int nhp_set_profiling(nhp_planner *p, int enable)
{
    if (!p) return NHP_E_ARG;
    DeviceGuard guard(p);
    if (enable && p->ev.empty() && !prof_grow(p)) return fail(p, NHP_E_CUDA, "creating the timing events failed");
    p->profiling = enable != 0;
    return NHP_OK;
}

int nhp_kernel_times(nhp_planner *p, double *ms_sum, long long *launches, int reset)
{
    if (!p) return NHP_E_ARG;
    DeviceGuard guard(p);
    CU(cudaStreamSynchronize(p->stream));
    for (int k = 0; k < p->ev_used; k++) {
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, p->ev[2 * k], p->ev[2 * k + 1]));
        p->k_ms[p->ev_slot[k]] += ms;
        p->k_launches[p->ev_slot[k]] += 1;
    }
    p->ev_used = 0;
    for (int s = 0; s < NHP_KERNEL_SLOTS; s++) {
        if (ms_sum) ms_sum[s] = p->k_ms[s];
        if (launches) launches[s] = p->k_launches[s];
        if (reset) { p->k_ms[s] = 0; p->k_launches[s] = 0; }
    }
    return NHP_OK;
}

}  // extern "C"
