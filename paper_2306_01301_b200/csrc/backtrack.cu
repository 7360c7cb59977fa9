// Back-tracking.  PAPER.md:376-382 (section X): "Each step of back-tracking is
// doing a Bellman-iteration in reverse ... back-tracing through all the maneuver curves that go through
// the current vertex in their entirety ... adding edge values sequentially and comparing the running sum
// plus the value of each vertex to the minimum so far", eq (32) l.380.  It is "like running the maneuver
// kernel in reverse, but for only one curve for each maneuver" -- so one block does it: warp m walks the
// curve of maneuver m through the current vertex, 32 vertices per step (addresses come straight from
// the curve maps (18)/(23), so nothing in the walk is a dependent load), with a warp prefix sum for E_sum
// and a warp arg-min.  Tie rule DESIGN R19: earliest maneuver in cycle order, then nearest source.
#include "nhp_internal.cuh"

struct BtParams {
    uint32_t ct[6];
    int log2_n, nt, fwd_only, soft;
    int si, sj, st, gi, gj, gt;
    int cap;
    int m0;                 // maneuver in progress at the start (-1: none): its segment out of the START carries no c_t
    int goal_from_status;   // the goal vertex comes from goal_search_kernel (status[4..6], found flag status[10])
};

__device__ __forceinline__ unsigned long long warp_min_u64(unsigned long long x)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const unsigned long long y = __shfl_xor_sync(0xffffffffu, x, d);
        x = y < x ? y : x;
    }
    return x;
}

__global__ void __launch_bounds__(192) backtrack_kernel(const uint32_t *__restrict__ V, const uint8_t *__restrict__ S,
                                                       DevTables T, BtParams P, nhp_waypoint *__restrict__ plan,
                                                       int32_t *__restrict__ status)
{
    __shared__ unsigned long long s_key[6];     // (candidate cost << 13) | steps back
    __shared__ uint32_t s_seg[6];               // ct + E_sum of the winning candidate
    __shared__ int s_cell[6][3];
    __shared__ int s_cur[4];                    // i, j, theta, continue flag
    const int m = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int log2_n = P.log2_n, n = 1 << log2_n, mx = n - 1, nt = P.nt, mt = nt - 1, quarter = nt >> 2;
    const unsigned long long KINF = ~0ull;
    int cnt = 0;
    unsigned long long total = 0;
    if (threadIdx.x == 0) {
        int go = 1;
        if (P.goal_from_status) { P.gi = status[4]; P.gj = status[5]; P.gt = status[6]; }
        const size_t gidx = ((((size_t)P.gt << log2_n) + P.gj) << log2_n) + P.gi;
        if (status[0]) { status[1] = NHP_E_START_BLOCKED; go = 0; }
        else if (P.goal_from_status && !status[10]) { status[1] = NHP_E_GOAL_UNREACHED; go = 0; }
        else if (V[gidx] == 0u) { status[1] = NHP_E_GOAL_UNREACHED; go = 0; }
        else if (P.gi == P.si && P.gj == P.sj && P.gt == P.st) {
            if (P.cap < 1) status[1] = NHP_E_BUFFER;
            else { plan[0] = nhp_waypoint{P.gi, P.gj, P.gt, -1}; status[1] = NHP_OK; status[2] = 1; status[3] = 0; }
            go = 0;
        }
        s_cur[0] = P.gi; s_cur[1] = P.gj; s_cur[2] = P.gt; s_cur[3] = go;
    }
    __syncthreads();
    while (s_cur[3]) {
        const int ci = s_cur[0], cj = s_cur[1], cth = s_cur[2];
        const bool turn = !(m == M_SF || m == M_SB);
        const bool skip = P.fwd_only && (m == M_RB || m == M_SB || m == M_LB);
        unsigned long long best = KINF;
        uint32_t best_seg = 0;
        int bi = 0, bj = 0, bt = 0;
        if (!skip) {
            // thread coordinates of the curve through the current vertex: inverse of (18) / (23), eq (29)
            int xp, yp, qa = 0, qb = 0, up;
            const int16_t *Bt = T.B + (size_t)cth * n;
            const int I = T.IJ[cth] & 1, jpos = (T.IJ[cth] >> 1) & 1;
            if (turn) {
                const bool left = (m == M_LF || m == M_LB);
                qa = left ? 0 : 2; qb = left ? 3 : 1;
                xp = (ci - T.beta[(cth + qa * quarter) & mt]) & mx;
                yp = (cj - T.beta[(cth + qb * quarter) & mt]) & mx;
                up = (m == M_LF || m == M_RB);
            } else {
                yp = I ? cj : ci;
                xp = ((I ? ci : cj) - Bt[yp]) & mx;
                up = ((m == M_SF) == (jpos == 1));
            }
            const int maxk = turn ? nt - 1 : n;
            const uint32_t ct = P.ct[m];
            // vertex k steps back, against the direction of m
            auto cell = [&](int k, int &i, int &j, int &t) {
                if (turn) {
                    t = (up ? cth - k : cth + k) & mt;
                    i = (xp + T.beta[(t + qa * quarter) & mt]) & mx;
                    j = (yp + T.beta[(t + qb * quarter) & mt]) & mx;
                } else {
                    const int y = (up ? yp - k : yp + k) & mx;
                    const int c = (xp + Bt[y]) & mx;
                    t = cth; i = I ? c : y; j = I ? y : c;
                }
            };
            unsigned long long E = 0;
            bool done = false;
            constexpr int NB = 8;                              // chunks of 32 vertices whose loads are in flight together
            for (int base = 0; base < maxk && !done; base += 32 * NB) {
                uint32_t uu[NB], ww[NB];
                bool at_start[NB];
#pragma unroll
                for (int c = 0; c < NB; c++) {
                    const int k = base + 32 * c + lane + 1;
                    int i, j, t;
                    cell(k, i, j, t);
                    const size_t idx = ((((size_t)t << log2_n) + j) << log2_n) + i;
                    const bool valid = k <= maxk;
                    uu[c] = valid ? V[idx] : 0u;
                    at_start[c] = (i == P.si && j == P.sj && t == P.st);
                    uint32_t w = T.len_q[(size_t)m * nt + t];
                    if (P.soft) w = (w * (uint32_t)(valid ? S[idx] : 16)) >> 4;
                    ww[c] = w;
                }
#pragma unroll
                for (int c = 0; c < NB; c++) {
                    if (done) continue;                          // warp-uniform
                    const int k = base + 32 * c + lane + 1;
                    const uint32_t u = uu[c];
                    const unsigned blk = __ballot_sync(0xffffffffu, u == 0u);       // blocked (or past the end)
                    const int first = blk ? __ffs(blk) - 1 : 32;
                    // inclusive prefix sum of the 32 edge weights of the chunk (each < 2^26: no wrap in 32 bits), then the running total
                    uint32_t p32 = (lane < first) ? ww[c] : 0u;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const uint32_t y = __shfl_up_sync(0xffffffffu, p32, d);
                        if (lane >= d) p32 += y;
                    }
                    const unsigned long long pre = E + p32;
                    if (lane < first && u < VI_INF) {
                        // u == 1 (cost 0) only at the start vertex: the maneuver in progress there is entered for free
                        const uint32_t ctm = (m == P.m0 && u == 1u && at_start[c]) ? 0u : ct;
                        const unsigned long long cand = (unsigned long long)(u - 1u) + ctm + pre;
                        if (cand < NHP_COST_LIMIT) {
                            // every lane keeps its own best; (cost, steps back) is the key, so the warp-wide minimum taken once at the
                            // end is the nearest source of least cost (DESIGN R19) whatever chunk it came from
                            const unsigned long long key = (cand << 13) | (unsigned)k;
                            if (key < best) { best = key; best_seg = (uint32_t)(ctm + pre); }
                        }
                    }
                    E += __shfl_sync(0xffffffffu, p32, 31);
                    if (first < 32) done = true;
                }
            }
            {
                const unsigned long long kmin = warp_min_u64(best);
                const unsigned who = __ballot_sync(0xffffffffu, best == kmin);
                best_seg = __shfl_sync(0xffffffffu, best_seg, __ffs(who) - 1);
                best = kmin;
            }
            if (best != KINF) cell((int)(best & 0x1fffu), bi, bj, bt);
        }
        if (lane == 0) { s_key[m] = best; s_seg[m] = best_seg; s_cell[m][0] = bi; s_cell[m][1] = bj; s_cell[m][2] = bt; }
        __syncthreads();
        if (threadIdx.x == 0) {
            int bm = -1;
            unsigned long long bc = KINF;
            for (int q = 0; q < 6; q++) {
                const unsigned long long c = s_key[q] == KINF ? KINF : (s_key[q] >> 13);
                if (c < bc) { bc = c; bm = q; }
            }
            if (bm < 0) { status[1] = NHP_E_GOAL_UNREACHED; s_cur[3] = 0; }
            else if (cnt >= P.cap) { status[1] = NHP_E_BUFFER; s_cur[3] = 0; }
            else {
                plan[cnt++] = nhp_waypoint{ci, cj, cth, bm};
                total += s_seg[bm];
                s_cur[0] = s_cell[bm][0]; s_cur[1] = s_cell[bm][1]; s_cur[2] = s_cell[bm][2];
                if (s_cur[0] == P.si && s_cur[1] == P.sj && s_cur[2] == P.st) {
                    if (cnt >= P.cap) status[1] = NHP_E_BUFFER;
                    else {
                        plan[cnt++] = nhp_waypoint{P.si, P.sj, P.st, -1};
                        status[1] = NHP_OK; status[2] = cnt;
                        status[3] = (int32_t)(total >= NHP_COST_LIMIT ? NHP_INF : (uint32_t)total);
                    }
                    s_cur[3] = 0;
                }
            }
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// Goal search, step 6 of the pipeline (section IX l.372-374; parameters d, W, w of appendix G l.1169):
// "more than one configuration in the goal set and ... a reward function ... over them.  The optimization criterion is
// the reward for the vertex minus the cost to get there ... Multiple ideal goals is also possible ... done on the GPU to
// avoid transferring the value volume".  Reading DESIGN R20: goal set = disc of radius d cells around the ideal pose
// times |dTheta| <= d, clipped at the grid border; criterion min V + W (di^2 + dj^2) + w dTheta^2; ties to the first
// candidate in the order (goal, dTheta, dj, di).  One block; key = (score << 24) | order, 64-bit min.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) goal_search_kernel(const uint32_t *__restrict__ V, const int32_t *__restrict__ goals, int n_goals,
                                                         int d, uint32_t W, uint32_t w, int log2_n, int nt, int32_t *__restrict__ status)
{
    __shared__ unsigned long long s_min[32];
    const int n = 1 << log2_n, side = 2 * d + 1, per_goal = side * side * side, total = n_goals * per_goal;
    unsigned long long best = ~0ull;
    for (int c = threadIdx.x; c < total; c += blockDim.x) {
        const int g = c / per_goal, r = c - g * per_goal;
        const int dt = r / (side * side) - d, dj = (r / side) % side - d, di = r % side - d;
        if (di * di + dj * dj > d * d) continue;
        const int i = goals[3 * g] + di, j = goals[3 * g + 1] + dj, t = (goals[3 * g + 2] + dt + 4 * nt) & (nt - 1);
        if (i < 0 || i >= n || j < 0 || j >= n) continue;
        const uint32_t v = V[((((size_t)t << log2_n) + j) << log2_n) + i];
        if (v == 0u || v >= VI_INF) continue;                                  // blocked / unreached (internal encoding)
        const unsigned long long score = (unsigned long long)(v - 1u) + (unsigned long long)W * (unsigned)(di * di + dj * dj) +
                                         (unsigned long long)w * (unsigned)(dt * dt);
        const unsigned long long key = (score << 24) | (unsigned)c;
        best = key < best ? key : best;
    }
    best = warp_min_u64(best);
    if ((threadIdx.x & 31) == 0) s_min[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x < 32) {
        best = threadIdx.x < (blockDim.x >> 5) ? s_min[threadIdx.x] : ~0ull;
        best = warp_min_u64(best);
        if (threadIdx.x == 0) {
            status[10] = best != ~0ull;
            if (best != ~0ull) {
                const int c = (int)(best & 0xffffffu), g = c / per_goal, r = c - g * per_goal;
                status[4] = goals[3 * g] + r % side - d;
                status[5] = goals[3 * g + 1] + (r / side) % side - d;
                status[6] = (goals[3 * g + 2] + r / (side * side) - d + 4 * nt) & (nt - 1);
                status[7] = g;
                status[8] = (int32_t)((best >> 24) & 0xffffffffu);
                status[9] = (int32_t)(best >> 56);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Start state with a maneuver in progress (section XII: "if a maneuver is in progress, there should be no
// transition cost to start with that maneuver, which is easily accomplished by using the appropriate start
// configuration"; DESIGN R26): the vertices AHEAD of the start on the curve of m0 are seeded with the summed edge weights
// from the start (no c_t) up to the first blocked vertex, at most one lap.  One warp, 32 vertices per step, warp prefix
// sum; runs once per plan between the init kernel and the first sweep.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32) seed_in_progress_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ S, DevTables T,
                                                              int log2_n, int nt, int soft, int si, int sj, int st, int m)
{
    const int lane = threadIdx.x, n = 1 << log2_n, mx = n - 1, mt = nt - 1, quarter = nt >> 2;
    const bool turn = !(m == M_SF || m == M_SB);
    int xp, yp, qa = 0, qb = 0, up;
    const int16_t *Bt = T.B + (size_t)st * n;
    const int I = T.IJ[st] & 1, jpos = (T.IJ[st] >> 1) & 1;
    if (turn) {
        const bool left = (m == M_LF || m == M_LB);
        qa = left ? 0 : 2; qb = left ? 3 : 1;
        xp = (si - T.beta[(st + qa * quarter) & mt]) & mx;
        yp = (sj - T.beta[(st + qb * quarter) & mt]) & mx;
        up = (m == M_LF || m == M_RB);
    } else {
        yp = I ? sj : si;
        xp = ((I ? si : sj) - Bt[yp]) & mx;
        up = ((m == M_SF) == (jpos == 1));
    }
    auto cell = [&](int k, int &i, int &j, int &t) {           // vertex k steps AHEAD of the start, in the direction of m
        if (turn) {
            t = (up ? st + k : st - k) & mt;
            i = (xp + T.beta[(t + qa * quarter) & mt]) & mx;
            j = (yp + T.beta[(t + qb * quarter) & mt]) & mx;
        } else {
            const int y = (up ? yp + k : yp - k) & mx;
            const int c = (xp + Bt[y]) & mx;
            t = st; i = I ? c : y; j = I ? y : c;
        }
    };
    if (V[((((size_t)st << log2_n) + sj) << log2_n) + si] == 0u) return;       // blocked start: reported by the init kernel
    const int maxk = turn ? nt - 1 : n;
    unsigned long long E = 0;
    for (int base = 0; base < maxk; base += 32) {
        const int k = base + lane + 1;
        int i, j, t, pi, pj, pt;
        cell(k, i, j, t);
        cell(k - 1, pi, pj, pt);                               // the edge into vertex k is charged at its source, vertex k - 1
        const size_t idx = ((((size_t)t << log2_n) + j) << log2_n) + i, pidx = ((((size_t)pt << log2_n) + pj) << log2_n) + pi;
        const bool valid = k <= maxk;
        const uint32_t u = valid ? V[idx] : 0u;
        const unsigned blk = __ballot_sync(0xffffffffu, u == 0u);
        const int first = blk ? __ffs(blk) - 1 : 32;
        uint32_t w = T.len_q[(size_t)m * nt + pt];
        if (soft) w = (w * (uint32_t)S[pidx]) >> 4;
        unsigned long long pre = (lane < first) ? w : 0;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long y = __shfl_up_sync(0xffffffffu, pre, d);
            if (lane >= d) pre += y;
        }
        pre += E;
        if (lane < first && pre < NHP_COST_LIMIT && (uint32_t)pre + 1u < u) V[idx] = (uint32_t)pre + 1u;
        E = __shfl_sync(0xffffffffu, pre, 31);
        if (first < 32) break;
    }
}

int launch_seed_in_progress(nhp_planner *p, int m0)
{
    ProfScope prof(p, 8);
    const int soft = (p->S != nullptr && (p->w.flags & NHP_FLAG_SOFT)) ? 1 : 0;
    seed_in_progress_kernel<<<1, 32, 0, p->stream>>>(p->V, p->S, p->tables(), p->log2_n, p->nt, soft, p->start[0], p->start[1], p->start[2], m0);
    return 1;
}

int launch_goal_search(nhp_planner *p, int n_goals, int d, uint32_t W, uint32_t w)
{
    ProfScope prof(p, 9);
    goal_search_kernel<<<1, 1024, 0, p->stream>>>(p->V, p->d_goals, n_goals, d, W, w, p->log2_n, p->nt, p->d_status);
    return 1;
}

int launch_backtrack(nhp_planner *p, int gi, int gj, int gt)
{
    BtParams P;
    for (int m = 0; m < 6; m++) P.ct[m] = p->w.ct[m];
    P.log2_n = p->log2_n; P.nt = p->nt;
    P.fwd_only = (p->w.flags & NHP_FLAG_FORWARD_ONLY) ? 1 : 0;
    P.soft = (p->S != nullptr && (p->w.flags & NHP_FLAG_SOFT)) ? 1 : 0;
    P.si = p->start[0]; P.sj = p->start[1]; P.st = p->start[2];
    P.gi = gi; P.gj = gj; P.gt = gt;
    P.cap = p->plan_cap;
    P.goal_from_status = gi < 0;
    P.m0 = p->start_m0;
    ProfScope prof(p, 9);
    backtrack_kernel<<<1, 192, 0, p->stream>>>(p->V, p->S, p->tables(), P, p->d_plan, p->d_status);
    return 1;
}
