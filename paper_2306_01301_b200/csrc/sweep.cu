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

// Cycle driver, PAPER.md:392 + l.475.  FORWARD_ONLY keeps LF, SF, RF.
int launch_cycles(nhp_planner *p, int n_cycles)
{
    int launches = 0;
    const bool fwd_only = p->w.flags & NHP_FLAG_FORWARD_ONLY;
    for (int c = 0; c < n_cycles; c++)
        for (int m = 0; m < 6; m++) {
            if (fwd_only && (m == M_RB || m == M_SB || m == M_LB)) continue;
            launches += launch_maneuver_simple(p, m);
        }
    return launches;
}
