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

// Edge weights of a section.  Hard obstacles only: one warp-uniform weight.  Soft: w = (len_q * S[p]) >> 4 per
// vertex (DESIGN R18), S taken from the curve-major copy of the soft volume: 32 bytes per thread and section, read
// 16 at a time in every pass (an L1 hit after the first) so that they do not occupy registers between passes.
template <bool SOFT>
struct SecW {
    uint32_t len;          // hard: the edge weight itself; soft: len_q << 4
    const uint4 *sp;       // soft: S of the section's 32 vertices, vertex k in byte k
};

__device__ __forceinline__ uint4 ld_s16(const uint4 *p)
{
    uint4 q;
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(q.x), "=r"(q.y), "=r"(q.z), "=r"(q.w) : "l"(p));
    return q;
}

template <bool SOFT, int K>
__device__ __forceinline__ uint32_t sec_weight(const SecW<SOFT> &sw, const uint4 &q)
{
    if (!SOFT) return sw.len;
    const uint32_t word = ((K >> 2) & 3) == 0 ? q.x : ((K >> 2) & 3) == 1 ? q.y : ((K >> 2) & 3) == 2 ? q.z : q.w;
    return nhp_soft_weight(sw.len, word, K & 3);
}

__device__ __forceinline__ void checksum_add(unsigned long long &acc, uint32_t v, uint32_t one);

// Two chains per thread.  A section of L = 32 vertices is swept as two half-sections H0, H1 (in travel order) whose
// chains are independent: both are summarised from "infinity" at the same time, the carry into H1 follows from the
// carry into H0 and H0's summary, and both are applied at the same time.  A single chain issues one dependent
// min/max op every ~4 cycles; two interleaved chains keep the integer pipe fed from half as many warps (the
// Sections algebra of appendix D, one level further down).
template <int L, bool UP, bool SOFT, bool CS, bool GATE, int S = 0>
struct SecLoop {
    static constexpr int H = L / 2;
    static constexpr int ka = UP ? S : L - 1 - S;             // vertex S of H0
    static constexpr int kb = UP ? H + S : H - 1 - S;         // vertex S of H1
    // summary pass: each half entered with "infinity" (Sv of Insert 3); t is the value AT the
    // vertex before its own edge (nhp_arrive / nhp_gate), wp the pending weight of the vertex behind it; for soft
    // weights d sums the edge costs across the half (Sd)
    static __device__ __forceinline__ void summary(const uint32_t (&col)[L], const SecW<SOFT> &sw, uint4 qa, uint4 qb, uint32_t &ta,
                                                   uint32_t &wa, uint32_t &da, uint32_t &tb, uint32_t &wb, uint32_t &db,
                                                   unsigned long long &acc, uint32_t one)
    {
        if (SOFT && S == 0) { qa = ld_s16(sw.sp + (ka >> 4)); qb = ld_s16(sw.sp + (kb >> 4)); }
        const uint32_t ua = col[ka], ub = col[kb];
        if (CS) { checksum_add(acc, ua, one); checksum_add(acc, ub, one); }
        ta = nhp_arrive(ta, wa, ua);
        tb = nhp_arrive(tb, wb, ub);
        if (GATE) { ta = nhp_gate(ta, ua); tb = nhp_gate(tb, ub); }
        wa = sec_weight<SOFT, ka>(sw, qa);
        wb = sec_weight<SOFT, kb>(sw, qb);
        if (SOFT) {                                              // on the FMA pipe (IMAD with the parameter 1), not the ALU pipe
            asm("mad.lo.u32 %0, %1, %2, %0;" : "+r"(da) : "r"(wa), "r"(one));
            asm("mad.lo.u32 %0, %1, %2, %0;" : "+r"(db) : "r"(wb), "r"(one));
        }
        SecLoop<L, UP, SOFT, CS, GATE, S + 1>::summary(col, sw, qa, qb, ta, wa, da, tb, wb, db, acc, one);
    }
    // apply pass: the vertex keeps min(v, u), then the same step
    static __device__ __forceinline__ void apply(uint32_t (&col)[L], const SecW<SOFT> &sw, uint4 qa, uint4 qb, uint32_t ct, uint32_t &ta,
                                                 uint32_t &wa, uint32_t &tb, uint32_t &wb, unsigned long long &acc, uint32_t one)
    {
        if (SOFT && S == 0) { qa = ld_s16(sw.sp + (ka >> 4)); qb = ld_s16(sw.sp + (kb >> 4)); }
        const uint32_t ua = col[ka], ub = col[kb];
        ta = nhp_arrive(ta, (!SOFT && S == 0) ? 0u : wa, ua);
        tb = nhp_arrive(tb, (!SOFT && S == 0) ? 0u : wb, ub);
        col[ka] = nhp_keep(ta, ct, ua);
        col[kb] = nhp_keep(tb, ct, ub);
        if (CS) { checksum_add(acc, col[ka], one); checksum_add(acc, col[kb], one); }
        if (GATE) { ta = nhp_gate(ta, ua); tb = nhp_gate(tb, ub); }
        if (SOFT) { wa = sec_weight<SOFT, ka>(sw, qa); wb = sec_weight<SOFT, kb>(sw, qb); }
        SecLoop<L, UP, SOFT, CS, GATE, S + 1>::apply(col, sw, qa, qb, ct, ta, wa, tb, wb, acc, one);
    }
};
template <int L, bool UP, bool SOFT, bool CS, bool GATE>
struct SecLoop<L, UP, SOFT, CS, GATE, L / 2> {
    static __device__ __forceinline__ void summary(const uint32_t (&)[L], const SecW<SOFT> &, uint4, uint4, uint32_t &, uint32_t &, uint32_t &,
                                                   uint32_t &, uint32_t &, uint32_t &, unsigned long long &, uint32_t) {}
    static __device__ __forceinline__ void apply(uint32_t (&)[L], const SecW<SOFT> &, uint4, uint4, uint32_t, uint32_t &, uint32_t &, uint32_t &,
                                                 uint32_t &, unsigned long long &, uint32_t) {}
};

// carry into section `sec` of a closed curve cut into S (a power of two) sections, travel direction UP
// (sec -> sec+1) or down: fold the other sections once around the curve, starting from section sec itself.
// The (M, D) table is stored twice, [2 S][32], so that the walk around the ring is a plain stride (one LDS with
// an immediate offset and one DPX op per section).  M <= 2^31 - 1 and D <= 2^31, so c + D never wraps.
template <bool UP>
__device__ __forceinline__ uint32_t ripple_carry(const uint2 *sMD, int sec, int S, int lane)
{
    const uint2 *q = sMD + (UP ? sec : sec + S) * 32 + lane;
    uint32_t c = q->x;
#pragma unroll 8
    for (int r = 1; r < S; r++) {
        q += UP ? 32 : -32;
        const uint2 md = *q;
        c = __viaddmin_u32(c, md.y, md.x);
    }
    return c;
}

// The same walk with the loads four sections ahead of the fold (the soft kernel has the registers for it at this point; in the hard
// kernel this form measured slower: 139 -> 144 us per pair)
template <bool UP>
__device__ __forceinline__ uint32_t ripple_carry_ahead(const uint2 *sMD, int sec, int S, int lane)
{
    const uint2 *q = sMD + (UP ? sec : sec + S) * 32 + lane;
    constexpr int step = UP ? 32 : -32;
    uint32_t c = q->x;
    // four (M, D) pairs are fetched while the four before them are folded: the dependent chain is the DPX ops, not the loads
    uint2 cur[4];
#pragma unroll
    for (int i = 0; i < 4; i++) cur[i] = (1 + i < S) ? q[(1 + i) * step] : make_uint2(0xffffffffu, 0u);
    for (int r = 1; r < S; r += 4) {
        uint2 nxt[4];
#pragma unroll
        for (int i = 0; i < 4; i++) nxt[i] = (r + 4 + i < S) ? q[(r + 4 + i) * step] : make_uint2(0xffffffffu, 0u);
#pragma unroll
        for (int i = 0; i < 4; i++) c = __viaddmin_u32(c, cur[i].y, cur[i].x);      // padding (M = 2^32 - 1, D = 0) leaves c as it is
#pragma unroll
        for (int i = 0; i < 4; i++) cur[i] = nxt[i];
    }
    return c;
}

// Exact change detection: the 64-bit sums of a thread's 32 vertices before and after the passes differ iff a vertex
// improved (values only decrease).  The additions are IMAD.WIDE on the FMA pipe; the "after" sum sits INSIDE the last
// apply loop, in the issue slots the min/max pipe leaves free (it takes one warp instruction every other cycle); the
// "before" sum is taken up front because it also tells whether every vertex of the warp is blocked.  The multiplier 1 comes from the
// kernel parameters: ptxas turns a multiplication by a KNOWN 1 into ALU-pipe IADD3 / IADD3.X pairs.
__device__ __forceinline__ void checksum_add(unsigned long long &acc, uint32_t v, uint32_t one)
{
    asm("mad.wide.u32 %0, %1, %2, %0;" : "+l"(acc) : "r"(v), "r"(one));
}

// Soft costs: ONE chain per thread over its section of L = 32 vertices (the per-vertex weight already gives the integer and
// the multiplier pipe independent work next to the chain, and a second chain's state does not fit the 64 registers of a
// 512-thread tile).  The S bytes come from the tile-major copy of the soft volume (softlayout.cu): word j of a section holds
// the bytes of its vertices 4 j .. 4 j + 3 for one curve, the 32 curves of the tile next to each other, so a warp reads one
// 128-byte line per four vertices (sp points at this lane's word 0; the line of word j is 32 words further on).  The word
// after the current one is fetched four vertices ahead.
__device__ __forceinline__ uint32_t ld_s4(const uint32_t *p)
{
    uint32_t q;
    asm volatile("ld.global.nc.u32 %0, [%1];" : "=r"(q) : "l"(p));
    return q;
}

// The pointer plus (x >> 31) words.  Every value x this is used with is below 2^31, so nothing is added -- but the instruction
// scheduler cannot know that, and the loads through the returned pointer (and the weight arithmetic that hangs on them) cannot
// be hoisted above the point where x is known.  Without it the weights of a whole pass are formed during the pass before it
// and spilled (the tile itself takes half the 64 registers).
__device__ __forceinline__ const uint32_t *after_value(const uint32_t *p, uint32_t x)
{
    return p + (x >> 31);
}

template <int L, bool UP, bool CS, int S = 0>
struct SoftLoop {
    static constexpr int k = UP ? S : L - 1 - S;
    static constexpr int knext = UP ? S + 4 : L - 1 - (S + 4);          // first vertex of the following word, in travel order
    static __device__ __forceinline__ void summary(const uint32_t (&col)[L], const uint32_t *sp, uint32_t len4, uint32_t &t, uint32_t &w, uint32_t &d,
                                                   uint32_t q, uint32_t qn, unsigned long long &acc, uint32_t one)
    {
        if (S % 4 == 0) { q = qn; if (S + 4 < L) qn = ld_s4(sp + 32 * (knext >> 2)); }
        const uint32_t u = col[k];
        if (CS) checksum_add(acc, u, one);
        const uint32_t wk = nhp_soft_weight(len4, q, k & 3);
        t = nhp_gate(nhp_arrive(t, w, u), u);
        w = wk;
        asm("mad.lo.u32 %0, %1, %2, %0;" : "+r"(d) : "r"(w), "r"(one));      // on the FMA pipe (IMAD with the parameter 1)
        SoftLoop<L, UP, CS, S + 1>::summary(col, sp, len4, t, w, d, q, qn, acc, one);
    }
    static __device__ __forceinline__ void apply(uint32_t (&col)[L], const uint32_t *sp, uint32_t len4, uint32_t ct, uint32_t &t, uint32_t &w, uint32_t q,
                                                 uint32_t qn, unsigned long long &acc, uint32_t one)
    {
        if (S % 4 == 0) { q = qn; if (S + 4 < L) qn = ld_s4(sp + 32 * (knext >> 2)); }
        const uint32_t u = col[k];
        const uint32_t wk = nhp_soft_weight(len4, q, k & 3);
        t = nhp_arrive(t, w, u);
        col[k] = nhp_keep(t, ct, u);
        if (CS) checksum_add(acc, col[k], one);
        t = nhp_gate(t, u);
        w = wk;
        SoftLoop<L, UP, CS, S + 1>::apply(col, sp, len4, ct, t, w, q, qn, acc, one);
    }
};
template <int L, bool UP, bool CS>
struct SoftLoop<L, UP, CS, L> {
    static __device__ __forceinline__ void summary(const uint32_t (&)[L], const uint32_t *, uint32_t, uint32_t &, uint32_t &, uint32_t &, uint32_t, uint32_t,
                                                   unsigned long long &, uint32_t) {}
    static __device__ __forceinline__ void apply(uint32_t (&)[L], const uint32_t *, uint32_t, uint32_t, uint32_t &, uint32_t &, uint32_t, uint32_t,
                                                 unsigned long long &, uint32_t) {}
};

struct TurnPass { uint32_t w, ct; };      // w: edge weight (hard) or len_q << 4 (soft)

// One maneuver over the tile.  All values travel as a = v - ct (nhp_arrive): a summary M is the value arriving at
// the first vertex BEHIND the (half-)section, D the summed edge cost across it (>= D_CAP: a blocked vertex interrupts it).
// Two warp-uniform short cuts (the only data-dependent control flow of the sweeps; the result is the same):
//   all_blocked   every vertex of the warp's 32 curves x 32 planes is blocked (deep inside an obstacle of the
//                 configuration space, ~20 % of the warps in configs 3 and 4): the section passes nothing on
//                 (M = infinity, D = D_CAP) and has nothing to update
//   none_blocked  no vertex is blocked (~16 %): the chains run without the nhp_gate op
//   no_finite     (hard costs only) no vertex of the warp holds a finite value yet: the section generates nothing
//                 (M = infinity, D as always), and if no finite value arrives either, the apply pass has nothing to do
// Returns true iff the apply pass ran (the vertices may have changed).
template <int L, bool UP, bool SOFT, bool CS_AFTER, bool CS_BEFORE>
__device__ __forceinline__ bool turn_maneuver(uint32_t (&col)[L], SecW<SOFT> &sw, TurnPass pass, bool blocked_lo, bool blocked_hi,
                                              bool all_blocked, bool none_blocked, bool &no_finite, uint2 *sMD, int sec, int S, int lane,
                                              unsigned long long &after, unsigned long long &before, uint32_t one, bool &tile_idle)
{
    // The barrier of a maneuver also tells whether EVERY section of the tile is in one of the two "hands on nothing" states: then
    // nothing can arrive anywhere, the ring need not be walked, and (the tile being unchanged) the same holds for the maneuver
    // that follows in a pair (tile_idle, CTA-uniform)
    if (all_blocked) {
        const uint2 md = make_uint2(0x7fffffffu, D_CAP);
        sMD[sec * 32 + lane] = md;
        sMD[(sec + S) * 32 + lane] = md;
        tile_idle = __syncthreads_and(1) != 0;
        return false;
    }
    if (!SOFT && no_finite) {
        const bool ia = UP ? blocked_lo : blocked_hi, ib = UP ? blocked_hi : blocked_lo;
        const uint32_t dh = (uint32_t)(L / 2) * pass.w;
        const uint2 md = make_uint2(0x7fffffffu, (ia || ib) ? D_CAP : 2 * dh);
        sMD[sec * 32 + lane] = md;
        sMD[(sec + S) * 32 + lane] = md;
        tile_idle = __syncthreads_and(1) != 0;
        if (tile_idle) return false;
        uint32_t ta = ripple_carry<UP>(sMD, sec, S, lane);
        if (__all_sync(0xffffffffu, ta >= VI_INF)) return false;                 // nothing arrives: nothing changes
        // something arrives: the ordinary apply pass (M of H0 is infinite, so the carry into H1 is ta + D(H0))
        // (no summary pass has run on this tile yet -- neither this maneuver's nor, in a pair, the one before: it would have cleared
        // no_finite -- so the "before" sum of the change detection is still to be taken)
#pragma unroll
        for (int k = 0; k < L; k++) checksum_add(before, col[k], one);
        uint32_t tb = __viaddmin_u32(ta, ia ? D_CAP : dh, 0x7fffffffu), wa = pass.w, wb = pass.w;
        sw.len = pass.w;
        SecLoop<L, UP, SOFT, CS_AFTER, true>::apply(col, sw, make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0), pass.ct, ta, wa, tb, wb, after, one);
        no_finite = false;
        return true;
    }
    const bool ia = UP ? blocked_lo : blocked_hi, ib = UP ? blocked_hi : blocked_lo;     // H0, H1 in travel order
    sw.len = pass.w;
    uint32_t ta = VI_INF, tb = VI_INF, wa = SOFT ? 0u : pass.w, wb = wa, da = 0, db = 0;
    if (none_blocked) SecLoop<L, UP, SOFT, CS_BEFORE, false>::summary(col, sw, make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0), ta, wa, da, tb, wb, db, before, one);
    else SecLoop<L, UP, SOFT, CS_BEFORE, true>::summary(col, sw, make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0), ta, wa, da, tb, wb, db, before, one);
    if (!SOFT) da = db = (uint32_t)(L / 2) * pass.w;
    const uint32_t ma = __viaddmin_u32(ta, wa, 0x7fffffffu), mb = __viaddmin_u32(tb, wb, 0x7fffffffu);
    const uint32_t Da = ia ? D_CAP : da;
    // section = H0 then H1: (Da, ma) o (Db, mb) = (Da + Db, min(ma + Db, mb)), Insert 4 PAPER.md:935-939
    const uint2 md = make_uint2(__viaddmin_u32(ma, ib ? D_CAP : db, mb), (ia || ib) ? D_CAP : da + db);
    sMD[sec * 32 + lane] = md;
    sMD[(sec + S) * 32 + lane] = md;
    tile_idle = __syncthreads_and(0) != 0;                    // (0: this section may hand something on)
    ta = ripple_carry<UP>(sMD, sec, S, lane);                 // carry into H0
    tb = __viaddmin_u32(ta, Da, ma);                          // carry into H1: through H0, or from inside it
    // opaque copy of the weight: otherwise the per-vertex values of the summary pass are kept alive for the apply pass
    asm volatile("" : "+r"(sw.len));
    wa = wb = SOFT ? 0u : sw.len;
    if (none_blocked) SecLoop<L, UP, SOFT, CS_AFTER, false>::apply(col, sw, make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0), pass.ct, ta, wa, tb, wb, after, one);
    else SecLoop<L, UP, SOFT, CS_AFTER, true>::apply(col, sw, make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0), pass.ct, ta, wa, tb, wb, after, one);
    return true;
}

// The same maneuver with soft costs (single chain, see SoftLoop).  Short cut kept: all_blocked.
template <int L, bool UP, bool CS_AFTER, bool CS_BEFORE>
__device__ __forceinline__ bool turn_maneuver_soft(uint32_t (&col)[L], const uint32_t *sp, TurnPass pass, bool blocked_any, bool all_blocked, uint2 *sMD,
                                                   int sec, int S, int lane, unsigned long long &after, unsigned long long &before, uint32_t one,
                                                   uint32_t &t_last)
{
    if (all_blocked) {
        const uint2 md = make_uint2(0x7fffffffu, D_CAP);
        sMD[sec * 32 + lane] = md;
        sMD[(sec + S) * 32 + lane] = md;
        __syncthreads();
        return false;
    }
    constexpr int k0 = UP ? 0 : L - 1;
    const uint32_t len4 = pass.w;
    uint32_t t = VI_INF, w = 0u, d = 0u;
    const uint32_t *sa = after_value(sp, t_last);             // not before the previous maneuver's last chain value
    SoftLoop<L, UP, CS_BEFORE>::summary(col, sa, len4, t, w, d, 0u, ld_s4(sa + 32 * (k0 >> 2)), before, one);
    const uint2 md = make_uint2(__viaddmin_u32(t, w, 0x7fffffffu), blocked_any ? D_CAP : d);
    sMD[sec * 32 + lane] = md;
    sMD[(sec + S) * 32 + lane] = md;
    __syncthreads();
    t = ripple_carry_ahead<UP>(sMD, sec, S, lane);
    const uint32_t *sb = after_value(sp, t);                  // not before the carry is known
    w = 0u;
    SoftLoop<L, UP, CS_AFTER>::apply(col, sb, len4, pass.ct, t, w, 0u, ld_s4(sb + 32 * (k0 >> 2)), after, one);
    t_last = t;
    return true;
}

// Row addressing of a tile: so[t] = element index of the tile's first vertex in plane t (row base + first column).
// A tile whose 32 columns never cross the seam i = N-1 -> 0 ("!wraps", CTA-uniform) addresses vertex (t, lane) as
// (V + lane)[so[t]]: one IMAD.WIDE per vertex; otherwise the column is wrapped per lane (one add + one bit-select more).
template <int L, bool WRAPS>
__device__ __forceinline__ void tile_rows_load(uint32_t (&col)[L], const uint32_t *__restrict__ V, const uint32_t *so, int lane, uint32_t mx)
{
    unsigned long long Vl = (unsigned long long)(V + (WRAPS ? 0 : lane));
    asm volatile("" : "+l"(Vl));            // opaque per-thread base: address = one IMAD.WIDE (base + 4 * index)
    const uint4 *so4 = (const uint4 *)so;
#pragma unroll
    for (int q = 0; q < L / 4; q++) {
        const uint4 o = so4[q];
        const uint32_t oo[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
        for (int e = 0; e < 4; e++) {
            uint32_t idx = oo[e];
            if (WRAPS) idx = ((idx + (uint32_t)lane) & mx) | (idx & ~mx);
            asm volatile("ld.global.u32 %0, [%1];" : "=r"(col[4 * q + e]) : "l"(Vl + 4ull * idx));
        }
    }
}

template <int L, bool WRAPS>
__device__ __forceinline__ void tile_rows_store(const uint32_t (&col)[L], uint32_t *__restrict__ V, const uint32_t *so, int lane, uint32_t mx)
{
    unsigned long long Vl = (unsigned long long)(V + (WRAPS ? 0 : lane));
    asm volatile("" : "+l"(Vl));
    const uint4 *so4 = (const uint4 *)so;
#pragma unroll
    for (int q = 0; q < L / 4; q++) {
        const uint4 o = so4[q];
        const uint32_t oo[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
        for (int e = 0; e < 4; e++) {
            uint32_t idx = oo[e];
            if (WRAPS) idx = ((idx + (uint32_t)lane) & mx) | (idx & ~mx);
            asm volatile("st.global.u32 [%0], %1;" ::"l"(Vl + 4ull * idx), "r"(col[4 * q + e]) : "memory");
        }
    }
}

template <int L, int NPASS, bool UP0, bool SOFT>
__global__ void __launch_bounds__(1024, 1) turn_tile_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ Scurve,
                                                          const int16_t *__restrict__ beta, int log2_n, int nt, int qa, int qb,
                                                          TurnPass pa, TurnPass pb, uint32_t one, int fixed, int bx0, int by0)
{
    extern __shared__ __align__(16) uint32_t smem[];
    const int S = nt / L, mt = nt - 1, quarter = nt >> 2, mx = (1 << log2_n) - 1;
    uint32_t *so = smem;                                      // [nt] element index of the tile's first vertex in every plane
    uint2 *sMD = (uint2 *)(so + nt);                          // [2][2 S][32] (M, D) of every section (twice), one set per maneuver
    const int lane = threadIdx.x & 31, sec = threadIdx.x >> 5;
    const int bx = blockIdx.x + bx0;                          // (bx0, by0): first tile of the launch; (0, 0) and a full grid but for the
    const int x0 = bx << 5, yp = blockIdx.y + by0;            // very first LF of a plan, see launch_cycles
    // every warp fills in the rows of its own 32 planes: no CTA-wide barrier stands between the start of a tile and its loads
    int seam;
    {
        const int t = sec * L + lane;
        const int ba = beta[(t + qa * quarter) & mt], bb = beta[(t + qb * quarter) & mt];     // eq (18)
        const int c0 = (x0 + ba) & mx;
        so[t] = (uint32_t)((((t << log2_n) + ((yp + bb) & mx)) << log2_n) + c0);
        seam = (c0 > mx - 31);
    }
    SecW<false> sw;
    sw.len = 0;
    sw.sp = nullptr;
    // tile-major soft volume (softlayout.cu): tile (yp, x0 / 32) = nt / 4 lines of 32 words; this section's words 8 sec .. 8 sec + 7
    const uint32_t *sp = nullptr;
    if (SOFT) {
        sp = (const uint32_t *)Scurve + (((size_t)yp << (log2_n - 5)) + bx) * ((size_t)nt * 8) + (size_t)sec * (L / 4) * 32;
        if (lane < L / 4) asm volatile("prefetch.global.L1 [%0];" ::"l"(sp + lane * 32));       // the section's eight lines, needed after the tile
        sp += lane;
    }
    const bool wraps = __any_sync(0xffffffffu, seam) != 0;      // warp-uniform
    __syncwarp();
    uint32_t col[L];
    if (!wraps) tile_rows_load<L, false>(col, V, so + sec * L, lane, (uint32_t)mx);
    else tile_rows_load<L, true>(col, V, so + sec * L, lane, (uint32_t)mx);
    // blocked vertices never change, so "does a blocked vertex interrupt this half of my section" is decided once
    uint32_t lo = col[0], hi = col[L / 2];
#pragma unroll
    for (int k = 1; k + 1 < L / 2; k += 2) {
        lo = __vimin3_u32(lo, col[k], col[k + 1]);
        hi = __vimin3_u32(hi, col[L / 2 + k], col[L / 2 + k + 1]);
    }
    const bool blocked_lo = min(lo, col[L / 2 - 1]) == 0u, blocked_hi = min(hi, col[L - 1]) == 0u;
    // change detection: `before` is summed inside the first summary pass, `after` inside the last apply pass (checksum_add)
    unsigned long long before = 0, after = 0;
    // `fixed` (NHP_FLAG_FIXED_WORK / NHP_FLAG_NO_SHORTCUTS) switches the three short cuts off; fixed == 1 also stores every row: the same
    // instructions and bytes whatever the volume holds
    // Short-cut conditions (warp-uniform).  Hard costs: the minimum over (v - 1) with wrap-around (blocked 0 -> 2^32 - 1, unreached
    // -> 2^30, finite below) tells both "every vertex of the warp is blocked" and "no finite value in this warp yet"; four
    // independent chains.  Soft costs (no no_finite short cut): a max tree for "all blocked".
    bool all_blocked = false, no_finite = false;
    if (!fixed) {
        if (SOFT) {
            uint32_t top = col[0];
#pragma unroll
            for (int k = 1; k + 1 < L; k += 2) top = __vimax3_u32(top, col[k], col[k + 1]);
            all_blocked = __all_sync(0xffffffffu, max(top, col[L - 1]) == 0u);
        } else {
            uint32_t m0 = 0xffffffffu, m1 = m0, m2 = m0, m3 = m0;
#pragma unroll
            for (int k = 0; k < L; k += 4) {
                m0 = __viaddmin_u32(col[k], 0xffffffffu, m0);
                m1 = __viaddmin_u32(col[k + 1], 0xffffffffu, m1);
                m2 = __viaddmin_u32(col[k + 2], 0xffffffffu, m2);
                m3 = __viaddmin_u32(col[k + 3], 0xffffffffu, m3);
            }
            const uint32_t lowest = min(min(m0, m1), min(m2, m3));
            all_blocked = __all_sync(0xffffffffu, lowest == 0xffffffffu);
            no_finite = __all_sync(0xffffffffu, lowest >= VI_INF - 1u);
        }
    }
    const bool none_blocked = !SOFT && !fixed && __all_sync(0xffffffffu, !blocked_lo && !blocked_hi);
    bool ran_a, ran_last, tile_idle = false;
    if constexpr (SOFT) {
        const bool blocked_any = blocked_lo || blocked_hi;
        uint32_t t_last = 0u;
        ran_a = turn_maneuver_soft<L, UP0, NPASS == 1, true>(col, sp, pa, blocked_any, all_blocked, sMD, sec, S, lane, after, before, one, t_last);
        ran_last = ran_a;
        if (NPASS == 2)
            ran_last = turn_maneuver_soft<L, !UP0, true, false>(col, sp, pb, blocked_any, all_blocked, sMD + 2 * S * 32, sec, S, lane, after, before, one, t_last);
    } else {
        ran_a = turn_maneuver<L, UP0, false, NPASS == 1, true>(col, sw, pa, blocked_lo, blocked_hi, all_blocked, none_blocked, no_finite, sMD, sec, S,
                                                               lane, after, before, one, tile_idle);
        ran_last = ran_a;
        if (NPASS == 2 && !tile_idle)
            ran_last = turn_maneuver<L, !UP0, false, true, false>(col, sw, pb, blocked_lo, blocked_hi, all_blocked, none_blocked, no_finite,
                                                                  sMD + 2 * S * 32, sec, S, lane, after, before, one, tile_idle);
    }
    if (!ran_last) {                                          // the "after" sum lives in the last apply pass: take it here if that pass did not run
        after = before;
        if (NPASS == 2 && ran_a) {
            after = 0;
#pragma unroll
            for (int k = 0; k < L; k++) checksum_add(after, col[k], one);
        }
    }
    if (after != before || fixed == 1) {
        int row0 = sec * L;
        asm volatile("" : "+r"(row0));        // re-read the row table: keeping the addresses alive across the passes spills
        if (!wraps) tile_rows_store<L, false>(col, V, so + row0, lane, (uint32_t)mx);
        else tile_rows_store<L, true>(col, V, so + row0, lane, (uint32_t)mx);
    }
}

// Can the tile kernel serve this planner?  Needs N_theta = 32 S with S <= 32 (one CTA) and 32-bit element indices.
static int turn_tile_L(const nhp_planner *p)
{
    if (p->w.flags & NHP_FLAG_SIMPLE_KERNELS) return 0;
    if ((size_t)p->n * p->n * p->nt > ((size_t)1 << 32)) return 0;
    return p->nt <= 1024 ? 32 : 0;
}

// One launch = maneuver ma (and then mb, the opposite direction on the same curve family, if mb >= 0).
static int launch_turn_tile(nhp_planner *p, int L, int ma, int mb, int only_bx = -1, int only_by = -1)
{
    const int n = p->n, nt = p->nt, S = nt / L;
    const bool soft = p->S != nullptr;
    const bool left = (ma == M_LF || ma == M_LB);
    const int qa = left ? 0 : 2, qb = left ? 3 : 1;
    const bool up = (ma == M_LF || ma == M_RB);
    auto pass = [&](int m) {
        TurnPass t{0, 0};
        // turn edge length does not depend on Theta (l.334); soft kernels take len_q << 4 (nhp_soft_weight)
        if (m >= 0) { t.w = soft ? p->len_q[(size_t)m * nt] << 4 : p->len_q[(size_t)m * nt]; t.ct = p->w.ct[m]; }
        return t;
    };
    const TurnPass pa = pass(ma), pb = pass(mb);
    const uint8_t *Sc = left ? p->S_left : p->S_right;
    const int fixed = (p->w.flags & NHP_FLAG_FIXED_WORK) ? 1 : (p->w.flags & NHP_FLAG_NO_SHORTCUTS) ? 2 : 0;   // 1: no short cuts, store all; 2: no short cuts
    const bool one_tile = only_bx >= 0;
    const dim3 grid(one_tile ? 1 : n / 32, one_tile ? 1 : n), block(32 * S);
    const int bx0 = one_tile ? only_bx : 0, by0 = one_tile ? only_by : 0;
    const size_t smem = sizeof(uint32_t) * (size_t)nt + sizeof(uint2) * 4 * (size_t)S * 32;
    ProfScope prof(p, mb >= 0 ? 11 : ma);
#define NHP_TT(NP, UP, SO) turn_tile_kernel<32, NP, UP, SO><<<grid, block, smem, p->stream>>>(p->V, Sc, p->d_beta, p->log2_n, nt, qa, qb, pa, pb, 1u, fixed, bx0, by0)
#define NHP_TT2(NP, UP) do { if (soft) NHP_TT(NP, UP, true); else NHP_TT(NP, UP, false); } while (0)
    if (mb >= 0) { if (up) NHP_TT2(2, true); else NHP_TT2(2, false); }
    else { if (up) NHP_TT2(1, true); else NHP_TT2(1, false); }
#undef NHP_TT2
#undef NHP_TT
    return 1;
}

static int launch_straight(nhp_planner *p, int m)
{
    const int k = launch_straight_tile(p, m);
    return k ? k : launch_maneuver_simple(p, m);
}

// Launches of one inner cycle of the tile kernels, in the paper's order with the two fusions: forward only: LF, SF, RF; otherwise
// SF, RB+RF, SB, LB+(next cycle's LF).
static int launch_inner_cycle(nhp_planner *p, int L, bool fwd_only)
{
    int launches = 0;
    if (fwd_only) {
        launches += launch_turn_tile(p, L, M_LF, -1);
        launches += launch_straight(p, M_SF);
        launches += launch_turn_tile(p, L, M_RF, -1);
    } else {
        launches += launch_straight(p, M_SF);
        launches += launch_turn_tile(p, L, M_RB, M_RF);
        launches += launch_straight(p, M_SB);
        launches += launch_turn_tile(p, L, M_LB, M_LF);
    }
    return launches;
}

// Small grids are bound by launch overhead (30 launches of a few microseconds each at 64^3): the launches of one
// inner cycle are captured once, at creation, into a CUDA graph and replayed.  Captured on a private stream (the caller's may
// be the legacy default stream, which cannot be captured); every kernel argument is fixed at creation.
int build_cycle_graph(nhp_planner *p)
{
    const int L = turn_tile_L(p);
    if (L == 0 || (size_t)p->n * p->n * p->nt > ((size_t)1 << 26)) return NHP_OK;
    cudaStream_t cap = nullptr, user = p->stream;
    if (cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) != cudaSuccess) return NHP_E_CUDA;
    const bool was_profiling = p->profiling;
    p->profiling = false;
    p->stream = cap;
    bool ok = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    int kernels = 0;
    if (ok) {
        kernels = launch_inner_cycle(p, L, (p->w.flags & NHP_FLAG_FORWARD_ONLY) != 0);
        ok = cudaStreamEndCapture(cap, &p->cycle_graph) == cudaSuccess && p->cycle_graph != nullptr;
    }
    p->stream = user;
    p->profiling = was_profiling;
    if (ok) ok = cudaGraphInstantiate(&p->cycle_exec, p->cycle_graph, 0) == cudaSuccess;
    cudaStreamDestroy(cap);
    if (!ok) { cudaGetLastError(); return NHP_E_CUDA; }
    p->cycle_graph_kernels = kernels;
    return NHP_OK;
}

// Cycle driver, PAPER.md:392 + l.475: LF, SF, RB, RF, SB, LB per cycle.  FORWARD_ONLY keeps LF, SF, RF.
// With the tile kernel, RB+RF run as one launch and LB is fused with the LF of the NEXT cycle (same curve family,
// adjacent in the sequence), so the order of operations on every vertex is exactly the paper's.
int launch_cycles(nhp_planner *p, int n_cycles, bool fresh)
{
    int launches = 0;
    const bool fwd_only = p->w.flags & NHP_FLAG_FORWARD_ONLY;
    const int L = turn_tile_L(p);
    const bool graph = p->cycle_exec != nullptr && !p->profiling;
    auto inner = [&]() {
        if (graph && cudaGraphLaunch(p->cycle_exec, p->stream) == cudaSuccess) return p->cycle_graph_kernels;
        return launch_inner_cycle(p, L, fwd_only);
    };
    for (int c = 0; c < n_cycles; c++) {
        if (L == 0) {
            for (int m = 0; m < 6; m++) {
                if (fwd_only && (m == M_RB || m == M_SB || m == M_LB)) continue;
                launches += (m == M_SF || m == M_SB) ? launch_straight(p, m) : launch_maneuver_simple(p, m);
            }
        } else if (fwd_only) {
            launches += inner();
        } else {
            // The very first LF of a plan finds one finite vertex, the start: only the left-turn curve through it can change
            // (PAPER.md:392 step 5; eq (18) inverted gives its thread coordinates), so one tile is launched instead of N^2 / 32; and
            // the SF that follows finds one finite vertex per Theta plane, those of that curve: one band per slice (streaming
            // kernels).  Not with a maneuver in progress at the start (more seeds) and not in the fixed-work modes.
            const bool first_sparse = c == 0 && fresh && p->start_m0 < 0 && !(p->w.flags & (NHP_FLAG_FIXED_WORK | NHP_FLAG_NO_SHORTCUTS));
            int xp = 0, yp = 0;
            if (first_sparse) {
                const int mt = p->nt - 1, mx = p->n - 1, q = p->nt >> 2, th = p->start[2];
                xp = (p->start[0] - p->beta[th & mt]) & mx; yp = (p->start[1] - p->beta[(th + 3 * q) & mt]) & mx;
            }
            if (c == 0) launches += first_sparse ? launch_turn_tile(p, L, M_LF, -1, xp >> 5, yp) : launch_turn_tile(p, L, M_LF, -1);
            const bool last = c + 1 == n_cycles;
            if (!last && !(first_sparse && !graph)) launches += inner();
            else {
                if (first_sparse && !graph) { p->sparse_xp = xp; p->sparse_yp = yp; }
                launches += launch_straight(p, M_SF);
                p->sparse_xp = p->sparse_yp = -1;
                launches += launch_turn_tile(p, L, M_RB, M_RF);
                launches += launch_straight(p, M_SB);
                launches += last ? launch_turn_tile(p, L, M_LB, -1) : launch_turn_tile(p, L, M_LB, M_LF);
            }
        }
    }
    return launches;
}
