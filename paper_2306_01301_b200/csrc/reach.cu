// Reachability ("bit-vector") planner, appendix C of the paper.
// Cost = number of maneuvers: "the value of a vertex during maneuver processing can be represented by a single bit ...
// if the vertex can be reached in m maneuvers or less" (l.871).  One bit per pose, 32 poses per word, layout as the
// collision volume C: word (Theta N + j) N/32 + i/32, bit i % 32 (here 1 = reachable; the paper's bit is inverted).
// Level m + 1 = level m OR the sweeps of all maneuvers over level m (a Jacobi step, l.871); "the output reachability
// bit volumes are kept around to support back-tracking" (l.897).  Loop body = Insert 2 (l.873-878):
//     v |= L_m[cell];  v &= ~C[cell];  L_m+1[cell] |= v          (blocked vertices removed, DESIGN R10)
// One thread sweeps a WORD of 32 neighbouring curves over one SECTION of the curve (appendix D, l.903-952, in its
// bit form: a section passes on G = what it generates itself and lets through P = the curves without an obstacle in
// it); the sections of a curve sit in one CTA and exchange (G, P) through shared memory.  A word of curves meets a
// plane at an arbitrary bit offset: reads are funnel shifts of two aligned words, writes are atomicOr of the two parts.
#include "nhp_internal.cuh"

namespace {

__device__ __forceinline__ uint32_t win32(const uint32_t *__restrict__ row, int x, int mw)
{
    const int w0 = (x >> 5) & mw;
    return __funnelshift_r(row[w0], row[(w0 + 1) & mw], x & 31);
}

__device__ __forceinline__ void or32(uint32_t *__restrict__ row, int x, int mw, uint32_t v)
{
    const int w0 = (x >> 5) & mw, sh = x & 31;
    atomicOr(row + w0, v << sh);
    if (sh) atomicOr(row + ((w0 + 1) & mw), v >> (32 - sh));
}

// carry into section `sec` of a ring of S sections in travel order UP (sec -> sec + 1) or down: start from the section
// itself, fold the others once around: c = (c & P_k) | G_k
template <bool UP>
__device__ __forceinline__ uint32_t ring_carry(const uint2 *sGP, int stride, int sec, int S)
{
    uint32_t c = sGP[sec * stride].x;
    for (int r = 1; r < S; r++) {
        const uint2 gp = sGP[((UP ? sec + r : sec - r + S) % S) * stride];
        c = (c & gp.y) | gp.x;
    }
    return c;
}

// Both maneuvers of one turn family (LF + LB, or RB + RF: the same curves, opposite directions) from ONE pass over the
// planes: the PL planes of a section are looked up once, (r, c) = (level bits, collision bits) stay in registers, and
// both directions are summarised and applied from there.  do_up / do_dn select the maneuvers (forward-only vehicles).
template <int PL>
__global__ void __launch_bounds__(512, 2) reach_turn2_kernel(uint32_t *__restrict__ Lout, const uint32_t *__restrict__ Lin, const uint32_t *__restrict__ C,
                                   const int16_t *__restrict__ beta, int log2_n, int nt, int qa, int qb, int do_up, int do_dn)
{
    extern __shared__ uint2 sGP[];                            // [S][nw] (G_up, P), [S][nw] (G_dn, P), [nt] plane table
    const int n = 1 << log2_n, mx = n - 1, nw = n >> 5, mw = nw - 1, mt = nt - 1, quarter = nt >> 2;
    const int xl = threadIdx.x, wx = blockDim.x, xw = blockIdx.y * wx + xl, sec = threadIdx.y, S = blockDim.y, yp = blockIdx.x;
    uint2 *sDn = sGP + S * wx, *sRow = sDn + S * wx;
    for (int t = sec * wx + xl; t < nt; t += S * wx) {
        const int ba = beta[(t + qa * quarter) & mt], bb = beta[(t + qb * quarter) & mt];     // eq (18)
        sRow[t] = make_uint2((uint32_t)((t * n + ((yp + bb) & mx)) * nw), (uint32_t)(ba & mx));
    }
    __syncthreads();
    uint32_t r[PL], c[PL];
    uint32_t p = ~0u;
#pragma unroll
    for (int k = 0; k < PL; k++) {
        const uint2 rw = sRow[sec * PL + k];
        const int x = (32 * xw + (int)rw.y) & mx;
        c[k] = win32(C + rw.x, x, mw);
        r[k] = win32(Lin + rw.x, x, mw);
        p &= ~c[k];
    }
    uint32_t vu = 0, vd = 0;
#pragma unroll
    for (int k = 0; k < PL; k++) {
        vu = (vu | r[k]) & ~c[k];
        vd = (vd | r[PL - 1 - k]) & ~c[PL - 1 - k];
    }
    sGP[sec * wx + xl] = make_uint2(vu, p);
    sDn[sec * wx + xl] = make_uint2(vd, p);
    __syncthreads();
    vu = do_up ? ring_carry<true>(sGP + xl, wx, sec, S) : 0u;
    vd = do_dn ? ring_carry<false>(sDn + xl, wx, sec, S) : 0u;
    uint32_t fresh[PL];
#pragma unroll
    for (int k = 0; k < PL; k++) {
        vu = (vu | r[k]) & ~c[k];
        fresh[k] = do_up ? vu & ~r[k] : 0u;
    }
#pragma unroll
    for (int k = PL - 1; k >= 0; k--) {
        vd = (vd | r[k]) & ~c[k];
        if (do_dn) fresh[k] |= vd & ~r[k];
        if (fresh[k]) {
            const uint2 rw = sRow[sec * PL + k];
            or32(Lout + rw.x, (32 * xw + (int)rw.y) & mx, mw, fresh[k]);
        }
    }
}

// Straight maneuvers SF + SB in "rows" form: step = row y of the slice, line x' sits at column (x' + B(y)) & mask, eq (23)
// with I = 1.  Slices with I = 0 are handled in their transposed copies, where they have exactly this form.
// CTA = one slice x all words of x' x S sections of PL rows; both directions from one pass over the rows (as above).
// The direction of SF is that of growing y iff J(Theta) > 0 (eq (24)); do_rev = 0 drops SB.
template <int PL>
__global__ void __launch_bounds__(512, 2) reach_rows2_kernel(uint32_t *__restrict__ Lout, const uint32_t *__restrict__ Lin, const uint32_t *__restrict__ C,
                                   const int16_t *__restrict__ B, const uint8_t *__restrict__ IJ, const int16_t *__restrict__ tlist,
                                   int log2_n, int do_rev)
{
    extern __shared__ uint2 sGP[];                            // [S][nw] (G_up, P), [S][nw] (G_dn, P)
    const int n = 1 << log2_n, mx = n - 1, nw = n >> 5, mw = nw - 1;
    const int xl = threadIdx.x, wx = blockDim.x, xw = blockIdx.y * wx + xl, sec = threadIdx.y, S = blockDim.y, t = tlist[blockIdx.x];
    const bool fwd_up = ((IJ[t] >> 1) & 1) != 0;
    const bool do_up = fwd_up || do_rev, do_dn = !fwd_up || do_rev;
    const int16_t *Bt = B + (size_t)t * n;
    const size_t slice = (size_t)t * n * nw;
    uint2 *sDn = sGP + S * wx;
    uint32_t r[PL], c[PL];
    uint32_t p = ~0u;
#pragma unroll
    for (int k = 0; k < PL; k++) {
        const int y = sec * PL + k;
        const int x = (32 * xw + Bt[y]) & mx;
        c[k] = win32(C + slice + (size_t)y * nw, x, mw);
        r[k] = win32(Lin + slice + (size_t)y * nw, x, mw);
        p &= ~c[k];
    }
    uint32_t vu = 0, vd = 0;
#pragma unroll
    for (int k = 0; k < PL; k++) {
        vu = (vu | r[k]) & ~c[k];
        vd = (vd | r[PL - 1 - k]) & ~c[PL - 1 - k];
    }
    sGP[sec * wx + xl] = make_uint2(vu, p);
    sDn[sec * wx + xl] = make_uint2(vd, p);
    __syncthreads();
    // (a line is not a ring, but its first cell y' = 0 is wall in both octant classes, so nothing wraps around)
    vu = do_up ? ring_carry<true>(sGP + xl, wx, sec, S) : 0u;
    vd = do_dn ? ring_carry<false>(sDn + xl, wx, sec, S) : 0u;
    uint32_t fresh[PL];
#pragma unroll
    for (int k = 0; k < PL; k++) {
        vu = (vu | r[k]) & ~c[k];
        fresh[k] = do_up ? vu & ~r[k] : 0u;
    }
#pragma unroll
    for (int k = PL - 1; k >= 0; k--) {
        vd = (vd | r[k]) & ~c[k];
        if (do_dn) fresh[k] |= vd & ~r[k];
        if (fresh[k]) {
            const int y = sec * PL + k;
            or32(Lout + slice + (size_t)y * nw, (32 * xw + Bt[y]) & mx, mw, fresh[k]);
        }
    }
}

// 32 x 32 bit-block transpose of the listed slices: dst (row = i, bit = j) from src (row = j, bit = i); ACC: OR into dst.
// One warp per block, lane = row of the block.
template <bool ACC>
__global__ void reach_transpose_kernel(uint32_t *__restrict__ dst, const uint32_t *__restrict__ src, const int16_t *__restrict__ tlist, int log2_n)
{
    const int n = 1 << log2_n, nw = n >> 5, lane = threadIdx.x;
    const size_t slice = (size_t)tlist[blockIdx.z] * n * nw;
    const int r0 = (blockIdx.y * blockDim.y + threadIdx.y) << 5, wc = blockIdx.x;
    const uint32_t word = src[slice + (size_t)(r0 + lane) * nw + wc];
    // five butterfly stages (swap the off-diagonal j x j blocks of every 2j x 2j block between lanes l and l ^ j)
    uint32_t mine = word, msk = 0x0000ffffu;
#pragma unroll
    for (int j = 16; j > 0; j >>= 1) {
        const uint32_t other = __shfl_xor_sync(0xffffffffu, mine, j);
        if (lane & j) mine ^= ((other >> j) ^ mine) & msk;
        else mine ^= ((((mine >> j) ^ other) & msk) << j);
        msk ^= msk << (j >> 1);
    }
    uint32_t *d = dst + slice + (size_t)(32 * wc + lane) * nw + (r0 >> 5);
    if (ACC) { if (mine) *d |= mine; } else *d = mine;
}

__global__ void reach_init_kernel(uint32_t *__restrict__ L0, const uint32_t *__restrict__ C, size_t nwords, size_t start_idx, int32_t *__restrict__ status)
{
    const size_t w = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= nwords) return;
    uint32_t v = 0;
    if ((start_idx >> 5) == w) {
        const uint32_t bit = 1u << (start_idx & 31);
        const bool blocked = (C[w] & bit) != 0;
        status[0] = blocked ? 1 : 0;
        if (!blocked) v = bit;
    }
    L0[w] = v;
}

struct RbParams {
    int log2_n, nt, fwd_only, n_levels;
    int si, sj, st, gi, gj, gt, cap;
    size_t level_words;
};

// smallest level at which vertex idx is reachable, or -1
__device__ __forceinline__ int reach_level(const uint32_t *__restrict__ L, size_t level_words, int n_levels, size_t idx)
{
    for (int m = 0; m <= n_levels; m++)
        if ((L[(size_t)m * level_words + (idx >> 5)] >> (idx & 31)) & 1u) return m;
    return -1;
}

// Back-tracking over the level volumes (l.897): from the goal at its level k, the maneuvers in cycle order;
// warp m walks back along the curve of maneuver m until a blocked vertex and reports the first vertex reachable at
// <= k - 1 maneuvers; the first maneuver with a candidate wins (DESIGN R27).  One block of six warps.
__global__ void __launch_bounds__(192) reach_backtrack_kernel(const uint32_t *__restrict__ L, const uint32_t *__restrict__ C, DevTables T,
                                                             RbParams P, nhp_waypoint *__restrict__ plan, int32_t *__restrict__ status)
{
    __shared__ int s_steps[6];
    __shared__ int s_cur[5];                    // i, j, theta, continue flag, level
    const int m = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int log2_n = P.log2_n, n = 1 << log2_n, mx = n - 1, nt = P.nt, mt = nt - 1, quarter = nt >> 2;
    int cnt = 0, total = 0;
    if (threadIdx.x == 0) {
        int go = 1;
        const size_t gidx = ((((size_t)P.gt << log2_n) + P.gj) << log2_n) + P.gi;
        const int k = status[0] ? -1 : reach_level(L, P.level_words, P.n_levels, gidx);
        if (status[0]) { status[1] = NHP_E_START_BLOCKED; go = 0; }
        else if (k < 0) { status[1] = NHP_E_GOAL_UNREACHED; go = 0; }
        else if (k == 0) {
            if (P.cap < 1) status[1] = NHP_E_BUFFER;
            else { plan[0] = nhp_waypoint{P.gi, P.gj, P.gt, -1}; status[1] = NHP_OK; status[2] = 1; status[3] = 0; }
            go = 0;
        }
        total = k;
        s_cur[0] = P.gi; s_cur[1] = P.gj; s_cur[2] = P.gt; s_cur[3] = go; s_cur[4] = k;
    }
    __syncthreads();
    while (s_cur[3]) {
        const int ci = s_cur[0], cj = s_cur[1], cth = s_cur[2], k = s_cur[4];
        const bool turn = !(m == M_SF || m == M_SB);
        const bool skip = P.fwd_only && (m == M_RB || m == M_SB || m == M_LB);
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
        auto cell = [&](int s, int &i, int &j, int &t) {          // vertex s steps back, against the direction of m
            if (turn) {
                t = (up ? cth - s : cth + s) & mt;
                i = (xp + T.beta[(t + qa * quarter) & mt]) & mx;
                j = (yp + T.beta[(t + qb * quarter) & mt]) & mx;
            } else {
                const int y = (up ? yp - s : yp + s) & mx;
                const int c = (xp + Bt[y]) & mx;
                t = cth; i = I ? c : y; j = I ? y : c;
            }
        };
        int steps = 0;                                              // 0 = no candidate
        if (!skip) {
            const int maxk = turn ? nt - 1 : n;
            const uint32_t *Lk = L + (size_t)(k - 1) * P.level_words;
            for (int base = 0; base < maxk; base += 32) {
                const int s = base + lane + 1;
                int i, j, t;
                cell(s, i, j, t);
                const size_t idx = ((((size_t)t << log2_n) + j) << log2_n) + i;
                const bool valid = s <= maxk;
                const bool blk = !valid || ((C[idx >> 5] >> (idx & 31)) & 1u);
                const bool hit = valid && ((Lk[idx >> 5] >> (idx & 31)) & 1u);
                const unsigned bm = __ballot_sync(0xffffffffu, blk), hm = __ballot_sync(0xffffffffu, hit);
                const int fb = bm ? __ffs(bm) - 1 : 32, fh = hm ? __ffs(hm) - 1 : 32;
                if (fh < fb) { steps = base + fh + 1; break; }
                if (fb < 32) break;
            }
        }
        if (lane == 0) s_steps[m] = steps;
        __syncthreads();
        // every warp sees the winner: the first maneuver in cycle order with a candidate
        int bm = -1;
        for (int q = 0; q < 6; q++) if (bm < 0 && s_steps[q] > 0) bm = q;
        __syncthreads();
        if (bm == m && lane == 0) {                                 // the winning warp moves the cursor (its cell() is the right one)
            int i, j, t;
            cell(s_steps[m], i, j, t);
            s_cur[0] = i; s_cur[1] = j; s_cur[2] = t;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            if (bm < 0) { status[1] = NHP_E_GOAL_UNREACHED; s_cur[3] = 0; }
            else if (cnt >= P.cap) { status[1] = NHP_E_BUFFER; s_cur[3] = 0; }
            else {
                plan[cnt++] = nhp_waypoint{ci, cj, cth, bm};
                const size_t idx = ((((size_t)s_cur[2] << log2_n) + s_cur[1]) << log2_n) + s_cur[0];
                s_cur[4] = reach_level(L, P.level_words, P.n_levels, idx);
                if (s_cur[0] == P.si && s_cur[1] == P.sj && s_cur[2] == P.st) {
                    if (cnt >= P.cap) status[1] = NHP_E_BUFFER;
                    else {
                        plan[cnt++] = nhp_waypoint{P.si, P.sj, P.st, -1};
                        status[1] = NHP_OK; status[2] = cnt; status[3] = total;
                    }
                    s_cur[3] = 0;
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace

// Level volumes L_0 .. L_n (kept for back-tracking) plus three volumes for the slices with I = 0, which are
// swept in their transposed copies (Lt = transposed level m, Ct = transposed collision bits, Gt = what the straight
// sweeps newly reach there).  Returns an NHP_ code; *launches counts kernels and copies.
int launch_reach_run(nhp_planner *p, int si, int sj, int st, int n_levels, int *launches)
{
    const int n = p->n, nt = p->nt, nw = n / 32;
    const size_t W = (size_t)n * n * nt / 32;
    if (!p->r_levels || n_levels > p->lim.max_reach_levels) return NHP_E_BUFFER;      // volumes are carved from the workspace at creation
    const bool fwd_only = p->w.flags & NHP_FLAG_FORWARD_ONLY;
    const int nx = p->n_xslices, ny = nt - nx;
    const int trows = n / 32 < 8 ? n / 32 : 8;                  // 32 x 32 blocks per CTA of the transposition
    const dim3 tgrid(nw, n / 32 / trows, nx > 0 ? nx : 1), tblk(32, trows);
    // sweeps: 16 planes (rows) per thread, as many words of curves per CTA as fit 512 threads (sections of different words
    // do not talk to each other); a curve has at most 4096 planes / rows (nhp_planner_create), i.e. at most 256 sections
    auto geom = [&](int len, int &PL, dim3 &blk, int &wgrid, size_t &smem, int table) {
        PL = 16;
        const int S = len / PL;
        int wx = 512 / S; if (wx > nw) wx = nw; if (wx < 1) wx = 1;
        blk = dim3(wx, S); wgrid = nw / wx;
        smem = sizeof(uint2) * ((size_t)2 * wx * S + table);
    };
    int PLn, PLr, tw, rw; dim3 tblk2, rblk2; size_t t2smem, r2smem;
    geom(nt, PLn, tblk2, tw, t2smem, nt);
    geom(n, PLr, rblk2, rw, r2smem, 0);
    int k = 0;
    reach_init_kernel<<<(unsigned)((W + 255) / 256), 256, 0, p->stream>>>(p->r_levels, p->C, W, ((size_t)st * n + sj) * n + si, p->d_rstatus);
    if (nx > 0) reach_transpose_kernel<false><<<tgrid, tblk, 0, p->stream>>>(p->r_Ct, p->C, p->d_tlist, p->log2_n);
    k += 2;
    for (int m = 0; m < n_levels; m++) {
        ProfScope prof(p, 13);
        const uint32_t *Lin = p->r_levels + (size_t)m * W;
        uint32_t *Lout = p->r_levels + (size_t)(m + 1) * W;
        cudaMemcpyAsync(Lout, Lin, sizeof(uint32_t) * W, cudaMemcpyDeviceToDevice, p->stream);
        // turn maneuvers, eq (18): LEFT (beta0, beta3), RIGHT (beta2, beta1); LF, RB travel Theta+, LB, RF Theta- (eqs (25)-(28))
        reach_turn2_kernel<16><<<dim3(n, tw), tblk2, t2smem, p->stream>>>(Lout, Lin, p->C, p->d_beta, p->log2_n, nt, 0, 3, 1, !fwd_only);   // LF (+ LB)
        reach_turn2_kernel<16><<<dim3(n, tw), tblk2, t2smem, p->stream>>>(Lout, Lin, p->C, p->d_beta, p->log2_n, nt, 2, 1, !fwd_only, 1);   // RF (+ RB)
        k += 3;
        if (ny > 0) {
            reach_rows2_kernel<16><<<dim3(ny, rw), rblk2, r2smem, p->stream>>>(Lout, Lin, p->C, p->d_B, p->d_IJ, p->d_tlist + nx, p->log2_n, !fwd_only);
            k += 1;
        }
        if (nx > 0) {
            reach_transpose_kernel<false><<<tgrid, tblk, 0, p->stream>>>(p->r_Lt, Lin, p->d_tlist, p->log2_n);
            cudaMemsetAsync(p->r_Gt, 0, sizeof(uint32_t) * W, p->stream);
            reach_rows2_kernel<16><<<dim3(nx, rw), rblk2, r2smem, p->stream>>>(p->r_Gt, p->r_Lt, p->r_Ct, p->d_B, p->d_IJ, p->d_tlist, p->log2_n, !fwd_only);
            reach_transpose_kernel<true><<<tgrid, tblk, 0, p->stream>>>(Lout, p->r_Gt, p->d_tlist, p->log2_n);
            k += 4;
        }
    }
    p->r_n_levels = n_levels;
    *launches = k;
    return NHP_OK;
}

namespace {
// one thread per word of 32 poses: first level whose bit is set
__global__ void reach_count_kernel(uint8_t *__restrict__ K, const uint32_t *__restrict__ L, size_t W, int n_levels)
{
    const size_t w = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= W) return;
    uint32_t seen = 0;
    uint8_t k[32];
#pragma unroll
    for (int b = 0; b < 32; b++) k[b] = 255;
    for (int m = 0; m <= n_levels; m++) {
        const uint32_t fresh = L[(size_t)m * W + w] & ~seen;
        if (fresh) {
#pragma unroll
            for (int b = 0; b < 32; b++) if ((fresh >> b) & 1u) k[b] = (uint8_t)m;
            seen |= fresh;
        }
    }
    uint4 *out = (uint4 *)(K + 32 * w);
#pragma unroll
    for (int q = 0; q < 2; q++) {
        uint32_t x[4];
#pragma unroll
        for (int e = 0; e < 4; e++) { const int b = 16 * q + 4 * e; x[e] = k[b] | (k[b + 1] << 8) | (k[b + 2] << 16) | ((uint32_t)k[b + 3] << 24); }
        out[q] = make_uint4(x[0], x[1], x[2], x[3]);
    }
}
}  // namespace

int launch_reach_count(nhp_planner *p, uint8_t *K_dev)
{
    const size_t W = (size_t)p->n * p->n * p->nt / 32;
    reach_count_kernel<<<(unsigned)((W + 127) / 128), 128, 0, p->stream>>>(K_dev, p->r_levels, W, p->r_n_levels);
    return 1;
}

int launch_reach_backtrack(nhp_planner *p, int gi, int gj, int gt)
{
    RbParams P;
    P.log2_n = p->log2_n; P.nt = p->nt; P.n_levels = p->r_n_levels;
    P.fwd_only = (p->w.flags & NHP_FLAG_FORWARD_ONLY) ? 1 : 0;
    P.si = p->r_start[0]; P.sj = p->r_start[1]; P.st = p->r_start[2];
    P.gi = gi; P.gj = gj; P.gt = gt; P.cap = p->plan_cap;
    P.level_words = (size_t)p->n * p->n * p->nt / 32;
    ProfScope prof(p, 9);
    reach_backtrack_kernel<<<1, 192, 0, p->stream>>>(p->r_levels, p->C, p->tables(), P, p->d_rplan, p->d_rstatus);
    return 1;
}
