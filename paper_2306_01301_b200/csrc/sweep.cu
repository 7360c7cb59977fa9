// Kernel-style N-turn graph processing.
// PAPER.md:354-364 (section VIII.B: one "maneuver kernel" sweeps every curve of one maneuver, in place,
// with the transition-in cost), Inserts 3-5 l.922-949 (loop body and the Sections algebra), l.475 (cycle
// order LF, SF, RB, RF, SB, LB), eq (18) l.266 and eq (23) l.291 (curve maps), l.334 (edge lengths).
//
// Per-vertex step of every sweep (Insert 5, l.946-949, in the internal encoding of nhp_internal.cuh):
//     out = min(v, u)                      V[i] = min(v, u)
//     v   = min(v + w', u + ct + w')       v = min(v, u + ct) + cx * B[i]
// with w' = w (edge weight at the SOURCE vertex, DESIGN R7) or VI_BIG when the vertex is blocked (u == 0),
// so that nothing propagates through a blocked vertex ("removed", DESIGN R10).  The
// second line is one DPX instruction (VIADDMNMX.U32).  No addition can wrap: v <= u + ct + w' <= 2^31 + 2^27.
#include "nhp_internal.cuh"

__device__ __forceinline__ void relax_step(uint32_t u, uint32_t w, uint32_t ct, uint32_t &v, uint32_t &out)
{
    const bool blocked = (u == 0u);
    const uint32_t wp = blocked ? VI_BIG : w;
    const uint32_t e = blocked ? VI_BIG : u + ct + w;
    out = min(v, u);
    v = __viaddmin_u32(v, wp, e);
}

// ---------------------------------------------------------------------------------------------
// V <- blocked ? 0 : VI_INF ; V[start] <- 1 (cost 0).  PAPER.md:392 step 5 initial state; the collision
// bits gate every later sweep through this stamp.  One thread per four vertices.
// ---------------------------------------------------------------------------------------------
__global__ void init_volume_kernel(uint4 *__restrict__ V4, const uint32_t *__restrict__ C, size_t nquads, size_t start_idx,
                                   int32_t *__restrict__ status)
{
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nquads) return;
    const size_t idx = q * 4;
    const uint32_t bits = C[idx >> 5] >> (idx & 31);
    uint4 o;
    o.x = (bits & 1u) ? 0u : VI_INF;
    o.y = (bits & 2u) ? 0u : VI_INF;
    o.z = (bits & 4u) ? 0u : VI_INF;
    o.w = (bits & 8u) ? 0u : VI_INF;
    if ((start_idx >> 2) == q) {
        uint32_t *c = &o.x + (start_idx & 3);
        status[0] = (*c == 0u) ? 1 : 0;            // start vertex collides -> NHP_E_START_BLOCKED later
        if (*c != 0u) *c = 1u;
    }
    V4[q] = o;
}

// internal <-> canonical (NHP_INF on blocked / unreached) conversion, in place
__global__ void export_volume_kernel(uint4 *__restrict__ V4, const uint32_t *__restrict__ C, size_t nquads, int to_canonical)
{
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nquads) return;
    uint4 v = V4[q];
    uint32_t *e = &v.x;
    if (to_canonical) {
#pragma unroll
        for (int k = 0; k < 4; k++) e[k] = (e[k] == 0u || e[k] >= VI_INF) ? NHP_INF : e[k] - 1u;
    } else {
        const size_t idx = q * 4;
        const uint32_t bits = C[idx >> 5] >> (idx & 31);
#pragma unroll
        for (int k = 0; k < 4; k++) e[k] = ((bits >> k) & 1u) ? 0u : (e[k] == NHP_INF ? VI_INF : e[k] + 1u);
    }
    V4[q] = v;
}

int launch_init_volume(nhp_planner *p, int si, int sj, int st)
{
    const size_t nr = (size_t)p->n * p->n * p->nt, nq = nr / 4;
    const size_t sidx = ((size_t)st * p->n + sj) * p->n + si;
    ProfScope prof(p, 8);
    init_volume_kernel<<<(unsigned)((nq + 255) / 256), 256, 0, p->stream>>>((uint4 *)p->V, p->C, nq, sidx, p->d_status);
    return 1;
}

int launch_export_volume(nhp_planner *p, bool to_canonical)
{
    const size_t nr = (size_t)p->n * p->n * p->nt, nq = nr / 4;
    ProfScope prof(p, 8);
    export_volume_kernel<<<(unsigned)((nq + 255) / 256), 256, 0, p->stream>>>((uint4 *)p->V, p->C, nq, to_canonical ? 1 : 0);
    return 1;
}

// ---------------------------------------------------------------------------------------------
// Bring-up kernels: the paper's own mapping, one thread per curve.
// Turn: thread = (x', y'), sweep coordinate Theta, two laps (the first only warms up v), eq (18).
// ---------------------------------------------------------------------------------------------
template <bool SOFT>
__global__ void __launch_bounds__(128) turn_simple_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ S,
                                                         const int16_t *__restrict__ beta, const uint32_t *__restrict__ lenq,
                                                         uint32_t ct, int log2_n, int nt, int qa, int qb, int up)
{
    extern __shared__ int16_t sbeta[];
    for (int k = threadIdx.x; k < nt; k += blockDim.x) sbeta[k] = beta[k];
    __syncthreads();
    const int mx = (1 << log2_n) - 1, mt = nt - 1, quarter = nt >> 2;
    const int xp = blockIdx.x * blockDim.x + threadIdx.x, yp = blockIdx.y;
    uint32_t v = VI_INF;
    for (int lap = 0; lap < 2; lap++) {
        for (int s = 0; s < nt; s++) {
            const int t = up ? s : nt - 1 - s;
            const int ba = sbeta[(t + qa * quarter) & mt], bb = sbeta[(t + qb * quarter) & mt];
            const size_t idx = ((((size_t)t << log2_n) + ((yp + bb) & mx)) << log2_n) + ((xp + ba) & mx);
            const uint32_t u = V[idx];
            uint32_t w = lenq[t], out;
            if (SOFT) w = (w * (uint32_t)S[idx]) >> 4;
            relax_step(u, w, ct, v, out);
            if (lap == 1 && out != u) V[idx] = out;
        }
    }
}

// Straight: thread = (x', Theta), sweep coordinate y', one lap starting at the wall, eq (23); direction by J (eq 24).
template <bool SOFT>
__global__ void __launch_bounds__(128) straight_simple_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ S,
                                                             const int16_t *__restrict__ B, const uint8_t *__restrict__ IJ,
                                                             const uint32_t *__restrict__ lenq, uint32_t ct, int log2_n,
                                                             int is_forward)
{
    const int n = 1 << log2_n, mx = n - 1;
    const int xp = blockIdx.x * blockDim.x + threadIdx.x, t = blockIdx.y;
    const int I = IJ[t] & 1, jpos = (IJ[t] >> 1) & 1;
    const int up = (is_forward == jpos);
    const int16_t *Bt = B + (size_t)t * n;
    const uint32_t len = lenq[t];
    uint32_t v = VI_INF;
    for (int s = 0; s < n; s++) {
        const int y = up ? s : n - 1 - s;
        const int c = (xp + Bt[y]) & mx;
        const int i = I ? c : y, j = I ? y : c;
        const size_t idx = ((((size_t)t << log2_n) + j) << log2_n) + i;
        const uint32_t u = V[idx];
        uint32_t w = len, out;
        if (SOFT) w = (w * (uint32_t)S[idx]) >> 4;
        relax_step(u, w, ct, v, out);
        if (out != u) V[idx] = out;
    }
}

static int launch_maneuver_simple(nhp_planner *p, int m)
{
    const int n = p->n, nt = p->nt;
    const bool soft = p->S != nullptr && (p->w.flags & NHP_FLAG_SOFT);
    const uint32_t *lenq = p->d_lenq + (size_t)m * nt;
    const uint32_t ct = p->w.ct[m];
    const int threads = n < 128 ? n : 128;
    ProfScope prof(p, m);
    if (m == M_SF || m == M_SB) {
        dim3 grid(n / threads, nt);
        if (soft)
            straight_simple_kernel<true><<<grid, threads, 0, p->stream>>>(p->V, p->S, p->d_B, p->d_IJ, lenq, ct, p->log2_n, m == M_SF);
        else
            straight_simple_kernel<false><<<grid, threads, 0, p->stream>>>(p->V, p->S, p->d_B, p->d_IJ, lenq, ct, p->log2_n, m == M_SF);
    } else {
        const int left = (m == M_LF || m == M_LB);
        const int qa = left ? 0 : 2, qb = left ? 3 : 1;          // eq (18): LEFT (beta0, beta3), RIGHT (beta2, beta1)
        const int up = (m == M_LF || m == M_RB);                 // eq (25), (28): Theta+ ; (26), (27): Theta-
        dim3 grid(n / threads, n);
        const size_t smem = sizeof(int16_t) * nt;
        if (soft)
            turn_simple_kernel<true><<<grid, threads, smem, p->stream>>>(p->V, p->S, p->d_beta, lenq, ct, p->log2_n, nt, qa, qb, up);
        else
            turn_simple_kernel<false><<<grid, threads, smem, p->stream>>>(p->V, p->S, p->d_beta, lenq, ct, p->log2_n, nt, qa, qb, up);
    }
    return 1;
}

// ---------------------------------------------------------------------------------------------
// Turn sweeps, B200 version: a tile of 32 curves stays ON CHIP for both laps and, where the cycle order puts two
// opposite-direction maneuvers of the same curve family next to each other (RB -> RF, LB -> next cycle's LF,
// PAPER.md:475), for both maneuvers: one read of the volume serves four laps.
//
// Tile = 32 consecutive x' at one y' (eq (18): every Theta plane of the tile is one 128-byte row segment, shifted
// by beta).  The N_theta planes are cut into S = N_theta / L sections (the paper's "Sections", appendix D,
// PAPER.md:903-952, here inside one CTA): warp s keeps planes [sL, sL+L) of its 32 curves in REGISTERS.
//   pass 1  every warp sweeps its section from v = infinity and records (M, D): the value leaving the section
//           and the summed edge cost across it (>= VI_BIG if a blocked vertex interrupts it) -- (Sv, Sd) of
//           Insert 3, l.923-928
//   ripple  carry into section s = fold of the other sections' (M, D) once around the closed curve, starting
//           from section s itself (this is what the first of the paper's "two full loops" computes, l.356)
//   pass 3  every warp sweeps its section again from that carry and updates its registers (Insert 5, l.946-949)
// (min, saturating +) is associative (DESIGN R18), so the result is bit-identical to the sequential two laps.
// Rows are written back only by threads whose section changed.
// ---------------------------------------------------------------------------------------------
constexpr uint32_t D_CAP = 1u << 31;     // "a blocked vertex interrupts this section" as a summed edge cost

// One vertex of a sweep with the arriving value v, exactly the paper's line (Insert 5):
//     v = min(v, u + ct) + cx * B[i]
// with the edge weight "infinite" at a blocked vertex (u == 0).  One DPX instruction + one add on the chain.
__device__ __forceinline__ uint32_t chain_step(uint32_t v, uint32_t u, uint32_t w, uint32_t ct)
{
    return __viaddmin_u32(u, ct, v) + (u != 0u ? w : VI_BIG);
}

template <int L, bool UP>
__device__ __forceinline__ uint32_t section_summary(const uint32_t (&col)[L], uint32_t w, uint32_t ct)
{
    uint32_t v = VI_INF;
#pragma unroll
    for (int s = 0; s < L; s++) v = chain_step(v, col[UP ? s : L - 1 - s], w, ct);
    return v;
}

// Apply pass: the vertex keeps min(v, u); the value that travels on is the same chain step.
template <int L, bool UP>
__device__ __forceinline__ void section_apply(uint32_t (&col)[L], uint32_t w, uint32_t ct, uint32_t v, bool &changed)
{
#pragma unroll
    for (int s = 0; s < L; s++) {
        const int k = UP ? s : L - 1 - s;
        const uint32_t u = col[k];
        changed |= (v < u);                    // accumulates in a predicate: no register, no longer live range
        col[k] = min(v, u);
        v = chain_step(v, u, w, ct);
    }
}

// carry into section `sec` of a closed curve cut into S (a power of two) sections, travel direction UP
// (sec -> sec+1) or down: fold the other sections once around the curve, starting from section sec itself.
template <bool UP>
__device__ __forceinline__ uint32_t ripple_carry(const uint32_t *sM, const uint32_t *sD, int sec, int S, int lane)
{
    uint32_t c = sM[sec * 32 + lane];
#pragma unroll 1
    for (int r = 1; r < S; r++) {
        const int q = (UP ? sec + r : sec - r) & (S - 1);
        c = __viaddmin_u32(c, sD[q * 32 + lane], sM[q * 32 + lane]);
    }
    return c;
}

struct TurnPass { uint32_t w, ct; };

template <int L, int NPASS, bool UP0>
__global__ void __launch_bounds__(1024, 1) turn_tile_kernel(uint32_t *__restrict__ V, const int16_t *__restrict__ beta,
                                                          int log2_n, int nt, int qa, int qb, TurnPass pa, TurnPass pb)
{
    extern __shared__ uint32_t smem[];
    const int S = nt / L, mt = nt - 1, quarter = nt >> 2, mx = (1 << log2_n) - 1;
    uint2 *soff = (uint2 *)smem;                              // [nt] (row base index, first column) of the tile
    uint32_t *sM = smem + 2 * nt, *sD = sM + 2 * S * 32;      // [2][S][32] each
    const int lane = threadIdx.x & 31, sec = threadIdx.x >> 5;
    const int x0 = blockIdx.x << 5, yp = blockIdx.y;
    for (int t = threadIdx.x; t < nt; t += blockDim.x) {
        const int ba = beta[(t + qa * quarter) & mt], bb = beta[(t + qb * quarter) & mt];     // eq (18)
        soff[t] = make_uint2((uint32_t)((((t << log2_n) + ((yp + bb) & mx)) << log2_n)), (uint32_t)((x0 + ba) & mx));
    }
    __syncthreads();
    // The apply passes take their weight through an opaque copy: otherwise the compiler keeps the 32 per-vertex
    // edge weights of the summary pass alive for the apply pass (common sub-expression) and spills them.
    const uint32_t wa = pa.w, ctwa = pa.ct, wb = pb.w, ctwb = pb.ct;
    uint32_t wa2 = pa.w, wb2 = pb.w;
    asm volatile("" : "+r"(wa2), "+r"(wb2));
    uint32_t col[L];
#pragma unroll
    for (int k = 0; k < L; k++) {
        const uint2 o = soff[sec * L + k];
        col[k] = V[o.x + ((o.y + lane) & mx)];
    }
    // blocked vertices never change, so "does a blocked vertex interrupt my section" is decided once
    uint32_t lowest = col[0];
#pragma unroll
    for (int k = 1; k < L; k++) lowest = min(lowest, col[k]);
    const bool interrupted = (lowest == 0u);
    bool changed = false;
    sM[sec * 32 + lane] = section_summary<L, UP0>(col, wa, ctwa);
    sD[sec * 32 + lane] = interrupted ? D_CAP : (uint32_t)L * wa;
    __syncthreads();
    section_apply<L, UP0>(col, wa2, ctwa, ripple_carry<UP0>(sM, sD, sec, S, lane), changed);
    if (NPASS == 2) {
        uint32_t *sM2 = sM + S * 32, *sD2 = sD + S * 32;
        sM2[sec * 32 + lane] = section_summary<L, !UP0>(col, wb, ctwb);
        sD2[sec * 32 + lane] = interrupted ? D_CAP : (uint32_t)L * wb;
        __syncthreads();
        section_apply<L, !UP0>(col, wb2, ctwb, ripple_carry<!UP0>(sM2, sD2, sec, S, lane), changed);
    }
    if (changed) {
        int row0 = sec * L;
        asm volatile("" : "+r"(row0));        // recompute the addresses: keeping 64 of them alive across the passes spills
#pragma unroll
        for (int k = 0; k < L; k++) {
            const uint2 o = soff[row0 + k];
            V[o.x + ((o.y + lane) & mx)] = col[k];
        }
    }
}

// Can the tile kernel serve this planner?  Needs N_theta = 32 S with S <= 32 (one CTA) and 32-bit element indices.
static int turn_tile_L(const nhp_planner *p)
{
    if (p->w.flags & NHP_FLAG_SIMPLE_KERNELS) return 0;
    if (p->S != nullptr && (p->w.flags & NHP_FLAG_SOFT)) return 0;            // soft variant: simple kernels for now
    if ((size_t)p->n * p->n * p->nt > ((size_t)1 << 32)) return 0;
    return p->nt <= 1024 ? 32 : 0;
}

// One launch = maneuver ma (and then mb, the opposite direction on the same curve family, if mb >= 0).
static int launch_turn_tile(nhp_planner *p, int L, int ma, int mb)
{
    const int n = p->n, nt = p->nt, S = nt / L;
    const bool left = (ma == M_LF || ma == M_LB);
    const int qa = left ? 0 : 2, qb = left ? 3 : 1;
    const bool up = (ma == M_LF || ma == M_RB);
    auto pass = [&](int m) {
        TurnPass t{0, 0};
        if (m >= 0) { t.w = p->len_q[(size_t)m * nt]; t.ct = p->w.ct[m]; }       // turn edge length does not depend on Theta (l.334)
        return t;
    };
    const TurnPass pa = pass(ma), pb = pass(mb);
    const dim3 grid(n / 32, n), block(32 * S);
    const size_t smem = sizeof(uint32_t) * (2 * (size_t)nt + 4 * (size_t)S * 32);
    ProfScope prof(p, mb >= 0 ? 11 : ma);
#define NHP_TT(LL, NP, UP) turn_tile_kernel<LL, NP, UP><<<grid, block, smem, p->stream>>>(p->V, p->d_beta, p->log2_n, nt, qa, qb, pa, pb)
    if (mb >= 0) { if (up) NHP_TT(32, 2, true); else NHP_TT(32, 2, false); }
    else { if (up) NHP_TT(32, 1, true); else NHP_TT(32, 1, false); }
#undef NHP_TT
    return 1;
}

static int launch_straight(nhp_planner *p, int m)
{
    const int k = launch_straight_tile(p, m);
    return k ? k : launch_maneuver_simple(p, m);
}

// Cycle driver, PAPER.md:392 + l.475: LF, SF, RB, RF, SB, LB per cycle.  FORWARD_ONLY keeps LF, SF, RF.
// With the tile kernel, RB+RF run as one launch and LB is fused with the LF of the NEXT cycle (same curve family,
// adjacent in the sequence), so the order of operations on every vertex is exactly the paper's.
int launch_cycles(nhp_planner *p, int n_cycles)
{
    int launches = 0;
    const bool fwd_only = p->w.flags & NHP_FLAG_FORWARD_ONLY;
    const int L = turn_tile_L(p);
    for (int c = 0; c < n_cycles; c++) {
        if (L == 0) {
            for (int m = 0; m < 6; m++) {
                if (fwd_only && (m == M_RB || m == M_SB || m == M_LB)) continue;
                launches += (m == M_SF || m == M_SB) ? launch_straight(p, m) : launch_maneuver_simple(p, m);
            }
        } else if (fwd_only) {
            launches += launch_turn_tile(p, L, M_LF, -1);
            launches += launch_straight(p, M_SF);
            launches += launch_turn_tile(p, L, M_RF, -1);
        } else {
            if (c == 0) launches += launch_turn_tile(p, L, M_LF, -1);
            launches += launch_straight(p, M_SF);
            launches += launch_turn_tile(p, L, M_RB, M_RF);
            launches += launch_straight(p, M_SB);
            launches += (c + 1 < n_cycles) ? launch_turn_tile(p, L, M_LB, M_LF) : launch_turn_tile(p, L, M_LB, -1);
        }
    }
    return launches;
}
