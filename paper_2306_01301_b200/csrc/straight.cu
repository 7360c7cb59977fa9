// Straight sweeps SF / SB, B200 version.
// PAPER.md:271-302 (section V.C, eqs (19)-(24): the discretised lines of one Theta slice), l.294 (direction by
// J), l.356 (one lap, started at the wall), Insert 5 l.946-949 (loop body), l.366-370 (the coalescing problem the
// paper solves with transposed slices and that is solved here by staging tiles in shared memory).
//
// One WARP owns a band of 32 neighbouring lines x' in [X0, X0+32) of one slice and walks along them in tiles of
// 32 sweep steps, carrying the travelling value of its 32 lines in registers (thread = line):
//   * slices with I = 1 (straight_rows_kernel): step = j, i = (x' + B(j)) & mask: every step is one (misaligned)
//     128-byte row segment in which lane l's word already is line l's vertex; tiles live in registers;
//   * slices with I = 0 (straight_xl_kernel): step = i, j = (x' + B(i)) & mask, eq (23): the lines run along the
//     memory-fast axis; tiles are parallelograms of the slice, loaded row-wise into registers one tile ahead,
//     passed through a per-warp stage in shared memory and read line-wise from there.
// A vertex is written back only if its value improved.
#include "nhp_internal.cuh"

namespace {

// Global addresses are formed as (opaque 64-bit slice base) + 4 * (32-bit element offset): one IMAD.WIDE.  The base
// is made opaque once per warp so that the compiler keeps it in a register pair instead of re-deriving it from
// the kernel parameters at every row.
__device__ __forceinline__ void st_global(unsigned long long vbase, uint32_t off, uint32_t val)
{
    asm volatile("st.global.u32 [%0], %1;\n" ::"l"(vbase + 4ull * off), "r"(val) : "memory");
}
__device__ __forceinline__ uint4 ld_nc16(const uint8_t *p)
{
    uint4 q;
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(q.x), "=r"(q.y), "=r"(q.z), "=r"(q.w) : "l"(p));
    return q;
}

// The first SF of a plan (launch_cycles): the only finite vertices are those of the left-turn curve through the start, one per
// Theta plane, so in every slice only the line through that vertex can change and only its band is launched.  xp < 0: off.
struct StartCurve {
    int xp, yp, nt;                  // thread coordinates of the curve, eq (18) inverted at the start
    const int16_t *beta, *B;
};

// line x' of slice t (I = 0 or 1, eq (23) inverted) through the start curve's vertex in plane t
template <int I>
__device__ __forceinline__ int start_curve_line(const StartCurve &sc, int t, int log2_n)
{
    const int n = 1 << log2_n, mx = n - 1, mt = sc.nt - 1, q = sc.nt >> 2;
    const int i = (sc.xp + sc.beta[t & mt]) & mx, j = (sc.yp + sc.beta[(t + 3 * q) & mt]) & mx;      // eq (18), left family (beta0, beta3)
    return I ? (i - sc.B[(size_t)t * n + j]) & mx : (j - sc.B[(size_t)t * n + i]) & mx;
}

// Relax the 32 steps of a tile for this thread's line (Insert 5, internal encoding, in the form
// of nhp_arrive: the value travels as t = value AT the vertex minus ct, wp = the pending edge weight of the vertex
// behind it):   t = min(t + wp, u);  V[i] = min(t + ct, u);  t = infinity behind a blocked vertex.
// Soft: w = (len_q * S) >> 4 per vertex, S from the line-major copy of the soft volume (s0, s1: this line's 32 bytes).
template <bool UP, bool SOFT, int S = 0>
struct RelaxLoop {
    static __device__ __forceinline__ void run(uint32_t *line, uint32_t &t, uint32_t &wp, uint32_t w, uint32_t ct, const uint4 &s0,
                                               const uint4 &s1, uint32_t &cm)
    {
        constexpr int k = UP ? S : 31 - S;
        const uint32_t u = line[k];
        t = nhp_arrive(t, wp, u);
        const uint32_t out = nhp_keep(t, ct, u);
        if (out != u) cm |= 1u << k;                                  // out <= u always
        line[k] = out;
        t = nhp_gate(t, u);
        if (!SOFT) wp = w;                                            // (only the first step can be entered with another pending weight)
        if (SOFT) {
            const uint4 &q = (k < 16) ? s0 : s1;
            const uint32_t word = ((k >> 2) & 3) == 0 ? q.x : ((k >> 2) & 3) == 1 ? q.y : ((k >> 2) & 3) == 2 ? q.z : q.w;
            wp = nhp_soft_weight(w, word, k & 3);
        }
        RelaxLoop<UP, SOFT, S + 1>::run(line, t, wp, w, ct, s0, s1, cm);
    }
};
template <bool UP, bool SOFT>
struct RelaxLoop<UP, SOFT, 32> {
    static __device__ __forceinline__ void run(uint32_t *, uint32_t &, uint32_t &, uint32_t, uint32_t, const uint4 &, const uint4 &, uint32_t &) {}
};

// Warp-uniform short cut (data-dependent, same result): nothing finite travels into this tile on any of the 32 lines
// (t >= VI_INF; every such value acts alike) and no vertex of the tile holds a finite value (v - 1 wraps blocked
// vertices to 2^32 - 1 and is >= 2^30 for unreached ones): the relaxation cannot change anything.  Four independent
// min chains.
__device__ __forceinline__ bool tile_is_idle4(const uint32_t (&u)[32], uint32_t t)
{
    uint32_t m0 = 0xffffffffu, m1 = m0, m2 = m0, m3 = m0;
#pragma unroll
    for (int k = 0; k < 32; k += 4) {
        m0 = __viaddmin_u32(u[k], 0xffffffffu, m0);
        m1 = __viaddmin_u32(u[k + 1], 0xffffffffu, m1);
        m2 = __viaddmin_u32(u[k + 2], 0xffffffffu, m2);
        m3 = __viaddmin_u32(u[k + 3], 0xffffffffu, m3);
    }
    const uint32_t lowest = min(min(m0, m1), min(m2, m3));
    return __all_sync(0xffffffffu, t >= VI_INF && lowest >= VI_INF - 1u);
}

// ---------------------------------------------------------------------------------------------
// Slices with I = 0 (|tan| <= 1, eq (19)): the sweep step is the COLUMN i and line x' sits at row
// (x' + B(i)) & mask, eq (23): the lines run along the memory-fast axis, so "thread = line" needs a transposition
// (the problem the paper solves by storing these slices transposed, l.366-370).  A warp owns a band of 32
// neighbouring lines and walks along it in tiles of 32 columns; a tile is a parallelogram of the slice.
// ---------------------------------------------------------------------------------------------
// RelaxLoop over one half of a tile (16 columns: HALF = 0 -> columns 0..15, 1 -> 16..31), values in h[0..15]; cm receives the
// tile-wide bit of every improved column
template <bool UP, bool SOFT, int HALF, int S = 0>
struct RelaxHalf {
    static __device__ __forceinline__ void run(uint32_t (&h)[16], uint32_t &t, uint32_t &wp, uint32_t w, uint32_t ct, const uint4 &q, uint32_t &cm)
    {
        constexpr int j = UP ? S : 15 - S, k = 16 * HALF + j;
        const uint32_t u = h[j];
        t = nhp_arrive(t, wp, u);
        const uint32_t out = nhp_keep(t, ct, u);
        if (out != u) cm |= 1u << k;                                  // out <= u always
        h[j] = out;
        t = nhp_gate(t, u);
        if (SOFT) {
            const uint32_t word = ((j >> 2) & 3) == 0 ? q.x : ((j >> 2) & 3) == 1 ? q.y : ((j >> 2) & 3) == 2 ? q.z : q.w;
            wp = nhp_soft_weight(w, word, j & 3);
        }
        RelaxHalf<UP, SOFT, HALF, S + 1>::run(h, t, wp, w, ct, q, cm);
    }
};
template <bool UP, bool SOFT, int HALF>
struct RelaxHalf<UP, SOFT, HALF, 16> {
    static __device__ __forceinline__ void run(uint32_t (&)[16], uint32_t &, uint32_t &, uint32_t, uint32_t, const uint4 &, uint32_t &) {}
};

// One half of a staged tile: gather the thread's 16 columns, relax them unless nothing finite is there or arrives (warp-uniform,
// see tile_is_idle), put the improved ones back into the stage.  offs4: the half's four uint4 of stage byte offsets.
template <bool UP, bool SOFT, int HALF>
__device__ __forceinline__ void xl_half(char *row, const uint4 *offs4, uint32_t &t, uint32_t &wp, uint32_t w, uint32_t ct, const uint4 &q, uint32_t &cm,
                                        int fixed)
{
    uint32_t h[16];
    const uint4 *o4 = offs4 + 4 * HALF;
#pragma unroll
    for (int e = 0; e < 4; e++) {
        const uint4 o = o4[e];
        h[4 * e + 0] = *(const uint32_t *)(row + o.x);
        h[4 * e + 1] = *(const uint32_t *)(row + o.y);
        h[4 * e + 2] = *(const uint32_t *)(row + o.z);
        h[4 * e + 3] = *(const uint32_t *)(row + o.w);
    }
    if (!fixed) {
        uint32_t m0 = 0xffffffffu, m1 = m0, m2 = m0, m3 = m0;
#pragma unroll
        for (int k = 0; k < 16; k += 4) {
            m0 = __viaddmin_u32(h[k], 0xffffffffu, m0);
            m1 = __viaddmin_u32(h[k + 1], 0xffffffffu, m1);
            m2 = __viaddmin_u32(h[k + 2], 0xffffffffu, m2);
            m3 = __viaddmin_u32(h[k + 3], 0xffffffffu, m3);
        }
        const uint32_t lowest = min(min(m0, m1), min(m2, m3));
        if (__all_sync(0xffffffffu, t >= VI_INF && lowest >= VI_INF - 1u)) return;
    }
    uint32_t c = 0;
    RelaxHalf<UP, SOFT, HALF>::run(h, t, wp, w, ct, q, c);
    if (fixed == 1) c = 0xffffu << (16 * HALF);           // NHP_FLAG_FIXED_WORK: every vertex goes back
    cm |= c;
    if (__any_sync(0xffffffffu, c != 0u)) {
#pragma unroll
        for (int e = 0; e < 4; e++) {
            const uint4 o = o4[e];
            if ((c >> (16 * HALF + 4 * e + 0)) & 1u) *(uint32_t *)(row + o.x) = h[4 * e + 0];
            if ((c >> (16 * HALF + 4 * e + 1)) & 1u) *(uint32_t *)(row + o.y) = h[4 * e + 1];
            if ((c >> (16 * HALF + 4 * e + 2)) & 1u) *(uint32_t *)(row + o.z) = h[4 * e + 2];
            if ((c >> (16 * HALF + 4 * e + 3)) & 1u) *(uint32_t *)(row + o.w) = h[4 * e + 3];
        }
    }
}

constexpr int XL_PITCH = 33, XL_ROWS = 39;
constexpr int XL_DATA = XL_ROWS * XL_PITCH;                // 1287 words
constexpr int XL_STAGE = XL_DATA + 32 + 1;                 // + the 32 stage byte offsets of the columns; 1320 words = 5280 bytes
#ifndef XL_WARPS_V
#define XL_WARPS_V 1
#endif
#ifndef XL_MINB_V
#define XL_MINB_V 20
#endif

// gather / scatter the 32 columns of this thread's line from / to the staged tile: `row` points at the thread's stage row, offs4 at
// the table of the columns' byte offsets (dq_k rows down, k words across; warp-uniform, read four at a time)
__device__ __forceinline__ void xr_gather0(uint32_t (&u)[32], const char *row, const uint4 *offs4)
{
#pragma unroll
    for (int q = 0; q < 8; q++) {
        const uint4 o = offs4[q];
        u[4 * q + 0] = *(const uint32_t *)(row + o.x);
        u[4 * q + 1] = *(const uint32_t *)(row + o.y);
        u[4 * q + 2] = *(const uint32_t *)(row + o.z);
        u[4 * q + 3] = *(const uint32_t *)(row + o.w);
    }
}
__device__ __forceinline__ void xr_scatter0(const uint32_t (&u)[32], char *row, const uint4 *offs4, uint32_t cm)
{
#pragma unroll
    for (int q = 0; q < 8; q++) {
        const uint4 o = offs4[q];
        if ((cm >> (4 * q + 0)) & 1u) *(uint32_t *)(row + o.x) = u[4 * q + 0];
        if ((cm >> (4 * q + 1)) & 1u) *(uint32_t *)(row + o.y) = u[4 * q + 1];
        if ((cm >> (4 * q + 2)) & 1u) *(uint32_t *)(row + o.z) = u[4 * q + 2];
        if ((cm >> (4 * q + 3)) & 1u) *(uint32_t *)(row + o.w) = u[4 * q + 3];
    }
}

// tile word of a lane (api.cu: upload_tables): dq | rows << 8 | (bmin + dlo8) << 16.  LOG2N > 0: the grid size is a compile-time
// constant, so the rows are immediate offsets from one base address as long as no lane's rows run across the seam j = N-1 -> 0
// (warp-uniform test; the tiles that do, a few per cent, take the general path)
template <int LOG2N>
__device__ __forceinline__ void xl_tile_load(uint32_t (&nx)[XL_ROWS], unsigned long long Vt, uint32_t tw, int T, int X0, int lane, int log2_n)
{
    const int rows = (tw >> 8) & 63, base = (int)tw >> 16;
    if (LOG2N > 0) {
        constexpr uint32_t N = 1u << LOG2N;
        const uint32_t j0 = (uint32_t)(X0 + base) & (N - 1u);
        if (__all_sync(0xffffffffu, j0 + XL_ROWS <= N)) {
            unsigned long long a = Vt + 4ull * ((j0 << LOG2N) + (uint32_t)(32 * T + lane));
            asm volatile("" : "+l"(a));
#pragma unroll
            for (int r = 0; r < XL_ROWS; r++)
                if (r < 32 || r < rows) asm volatile("ld.global.u32 %0, [%1];" : "=r"(nx[r]) : "l"(a + (unsigned long long)r * (4ull << LOG2N)));
            return;
        }
    }
    const uint32_t smask = (1u << (2 * log2_n)) - 1u, rstep = 1u << log2_n;
    uint32_t off = ((((uint32_t)(X0 + base)) << log2_n) & smask) + (uint32_t)(32 * T + lane);
#pragma unroll
    for (int r = 0; r < XL_ROWS; r++) {
        if (r < 32 || r < rows) asm volatile("ld.global.u32 %0, [%1];" : "=r"(nx[r]) : "l"(Vt + 4ull * off));
        off = (off + rstep) & smask;
    }
}

// rows of the stage back to the volume: lane = column k; the element in stage row q belongs to line q - dq and is written if
// that line improved in this tile; only the rows between the first and the last improved line
__device__ __forceinline__ void xl_stage_store(const uint32_t *sp, unsigned long long Vt, uint32_t tw, int T, int X0, int lane, int log2_n,
                                               uint32_t lines)
{
    const uint32_t smask = (1u << (2 * log2_n)) - 1u, rstep = 1u << log2_n;
    const int dq = tw & 7, base = (int)tw >> 16;
    const unsigned long long want = (unsigned long long)lines << dq;
    const int q0 = __ffs(lines) - 1, q1 = 32 - __clz(lines) + 7;
    uint32_t off = ((((uint32_t)(X0 + base + q0)) << log2_n) & smask) + (uint32_t)(32 * T + lane);
    uint32_t wlo = (uint32_t)(want >> q0), whi = (uint32_t)((want >> q0) >> 32);
    const uint32_t *s = sp + q0 * XL_PITCH + lane;
    for (int q = q0; q < q1; q += 4) {                        // warp-uniform bounds
#pragma unroll
        for (int e = 0; e < 4; e++) {
            if ((wlo >> e) & 1u) st_global(Vt, off, s[e * XL_PITCH]);
            off = (off + rstep) & smask;
        }
        wlo = __funnelshift_r(wlo, whi, 4);
        whi >>= 4;
        s += 4 * XL_PITCH;
    }
}

template <bool SOFT, int LOG2N>
__global__ void __launch_bounds__(32 * XL_WARPS_V, XL_MINB_V) straight_xl_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ Sline,
                                                                               const uint32_t *__restrict__ xl_tab, const uint8_t *__restrict__ IJ,
                                                                               const int16_t *__restrict__ tlist, const uint32_t *__restrict__ lenq,
                                                                               uint32_t ct, int log2_n, int is_forward, int fixed, StartCurve sc)
{
    extern __shared__ __align__(16) uint32_t smem[];
    const int xs = blockIdx.y, t = tlist[xs];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int X0 = sc.xp >= 0 ? (start_curve_line<0>(sc, t, log2_n) & ~31) : (blockIdx.x * (blockDim.x >> 5) + warp) << 5;
    const bool up = (is_forward == ((IJ[t] >> 1) & 1));                         // eq (24)
    const int NT = 1 << (log2_n - 5);
    unsigned long long Vt = (unsigned long long)(V + ((size_t)t << (2 * log2_n)));
    asm volatile("" : "+l"(Vt));
    // S_line[Theta][band][T][half][lane][16] (softlayout.cu): this thread's line, two 16-byte pieces per tile, 1024 bytes from tile to tile
    const uint8_t *Sl = SOFT ? Sline + ((size_t)t << (2 * log2_n)) + (((size_t)(X0 >> 5) << (log2_n - 5)) << 10) + 16 * lane : nullptr;
    uint32_t *stage = smem + warp * XL_STAGE;
    char *row = (char *)(stage + lane * XL_PITCH);
    const uint4 *offs4 = (const uint4 *)(stage + XL_DATA + 1);                  // 16-byte aligned: XL_DATA + 1 = 1288
    const uint32_t *tab = xl_tab + (size_t)xs * NT * 32 + lane;
    const uint32_t w = SOFT ? lenq[t] << 4 : lenq[t];
    uint32_t nx[XL_ROWS];
    uint4 ns0 = make_uint4(0, 0, 0, 0), ns1 = ns0;
    int T = up ? 0 : NT - 1;
    uint32_t tw = tab[T * 32], tw_next = NT > 1 ? tab[(up ? 1 : NT - 2) * 32] : 0u;
    xl_tile_load<LOG2N>(nx, Vt, tw, T, X0, lane, log2_n);
    if (SOFT) { ns0 = ld_nc16(Sl + 1024 * T); ns1 = ld_nc16(Sl + 1024 * T + 512); }
    uint32_t tv = VI_INF, wp = SOFT ? 0u : w;          // nothing arrives at the wall cell the line starts from
#pragma unroll 1
    for (int s = 0; s < NT; s++) {
        __syncwarp();                                  // the stage is free (row stores of the previous tile have read it)
        const uint32_t tw_cur = tw;
        const int T_cur = T, rows = (tw >> 8) & 63;
        {
#pragma unroll
            for (int r = 0; r < XL_ROWS; r++)
                if (r < 32 || r < rows) stage[r * XL_PITCH + lane] = nx[r];
            stage[XL_DATA + 1 + lane] = (uint32_t)(((tw & 7) * XL_PITCH + lane) * 4);
        }
        const uint4 s0 = ns0, s1 = ns1;
        if (s + 1 < NT) {                              // the next tile into the registers the stage has just been filled from (no
            T = up ? s + 1 : NT - 2 - s;               // barrier in between: the loads go out as soon as the stores have read them)
            tw = tw_next;
            xl_tile_load<LOG2N>(nx, Vt, tw, T, X0, lane, log2_n);
            if (SOFT) { ns0 = ld_nc16(Sl + 1024 * T); ns1 = ld_nc16(Sl + 1024 * T + 512); }
            if (s + 2 < NT) tw_next = tab[(up ? s + 2 : NT - 3 - s) * 32];
        }
        __syncwarp();
        uint32_t cm = 0;
        if (up) {
            xl_half<true, SOFT, 0>(row, offs4, tv, wp, w, ct, s0, cm, fixed);
            xl_half<true, SOFT, 1>(row, offs4, tv, wp, w, ct, s1, cm, fixed);
        } else {
            xl_half<false, SOFT, 1>(row, offs4, tv, wp, w, ct, s1, cm, fixed);
            xl_half<false, SOFT, 0>(row, offs4, tv, wp, w, ct, s0, cm, fixed);
        }
        const uint32_t lines = __ballot_sync(0xffffffffu, cm != 0u);
        if (lines) {
            __syncwarp();
            xl_stage_store(stage, Vt, tw_cur, T_cur, X0, lane, log2_n, lines);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Slices with I = 1 (eq (19)): the sweep step is the ROW j and line x' sits at column
// (x' + B(j)) & mask, so a warp that owns 32 neighbouring lines reads, at every step, one (misaligned, possibly
// wrapping) 128-byte row segment in which lane l's word already IS line l's vertex: no transposition, no shared
// memory.  A tile of 32 steps lives in 32 registers per thread (plain LDG: 1.8 cycles per warp instruction against
// the 8 of a 4-byte cp.async, profiles/r01_tile_kernels.md); all warps of the launch are resident at once and the
// loads of one warp's tile overlap the chains of the others.  Vertices that improve are stored from the thread
// that owns them.
// ---------------------------------------------------------------------------------------------
template <bool SOFT>
__global__ void __launch_bounds__(128, 7) straight_rows_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ Sline,
                                                            const int16_t *__restrict__ B, const uint8_t *__restrict__ IJ,
                                                            const int16_t *__restrict__ tlist,
                                                            const uint32_t *__restrict__ lenq, uint32_t ct, int log2_n, int is_forward, int fixed,
                                                            StartCurve sc)
{
    const int n = 1 << log2_n, mx = n - 1, t = tlist[blockIdx.y];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // (sparse first SF: the CTA's four warps take the aligned group of four bands that holds the line)
    const int X0 = sc.xp >= 0 ? (((start_curve_line<1>(sc, t, log2_n) >> 5) & ~3) + warp) << 5 : (blockIdx.x * (blockDim.x >> 5) + warp) << 5;
    const int jpos = (IJ[t] >> 1) & 1;
    const bool up = (is_forward == jpos);                                       // eq (24)
    const int16_t *Bt = B + (size_t)t * n;
    unsigned long long Vt = (unsigned long long)(V + ((size_t)t << (2 * log2_n)));
    asm volatile("" : "+l"(Vt));
    const uint8_t *Sl = SOFT ? Sline + ((size_t)t << (2 * log2_n)) + (((size_t)(X0 >> 5) << (log2_n - 5)) << 10) + 16 * lane : nullptr;
    const uint32_t w = SOFT ? lenq[t] << 4 : lenq[t];
    const uint32_t c0 = (uint32_t)(X0 + lane);
    const int NT = n >> 5;
    uint32_t tv = VI_INF, wp = SOFT ? 0u : w;
#pragma unroll 1
    for (int s = 0; s < NT; s++) {
        const int T = up ? s : NT - 1 - s;
        const int bmine = Bt[32 * T + lane];
        const uint32_t row0 = (uint32_t)(32 * T) << log2_n;
        uint32_t u[32];
#pragma unroll
        for (int k = 0; k < 32; k++) {
            const int b = __shfl_sync(0xffffffffu, bmine, k);
            const uint32_t off = row0 + ((uint32_t)k << log2_n) + ((c0 + (uint32_t)b) & (uint32_t)mx);
            u[k] = *(const uint32_t *)(Vt + 4ull * off);
        }
        uint4 s0 = make_uint4(0, 0, 0, 0), s1 = s0;
        if (SOFT) { s0 = ld_nc16(Sl + 1024 * T); s1 = ld_nc16(Sl + 1024 * T + 512); }
        uint32_t cm = 0;
        if (!fixed && tile_is_idle4(u, tv)) { }
        else if (up) RelaxLoop<true, SOFT>::run(u, tv, wp, w, ct, s0, s1, cm);
        else RelaxLoop<false, SOFT>::run(u, tv, wp, w, ct, s0, s1, cm);
        if (fixed == 1) cm = 0xffffffffu;                       // NHP_FLAG_FIXED_WORK: every vertex goes back
        if (__any_sync(0xffffffffu, cm != 0u)) {
#pragma unroll
            for (int k = 0; k < 32; k++) {
                const int b = __shfl_sync(0xffffffffu, bmine, k);
                const uint32_t off = row0 + ((uint32_t)k << log2_n) + ((c0 + (uint32_t)b) & (uint32_t)mx);
                if ((cm >> k) & 1u) st_global(Vt, off, u[k]);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Sections for the straight sweeps (appendix D, Inserts 3-5): one CTA = one band of 32 neighbouring
// lines, one WARP = one section = one tile of 32 sweep steps, all tiles of the band resident at once.
//   pass 1  every warp sweeps its tile from v = infinity: (M, D) = the value arriving behind the tile and the summed edge cost
//           across it (>= D_CAP if a blocked vertex interrupts it) -- (Sv, Sd) of Insert 3, l.923-928
//   ripple  carry into section s = fold of the sections before it in travel order, (c, D, M) -> min(c + D, M), Insert 4
//           l.935-939; the first section starts from infinity (the wall cell, DESIGN R12)
//   pass 2  every warp sweeps its tile again from its carry (Insert 5, l.946-949)
// (min, saturating +) is associative (DESIGN R18): bit-identical to the walk of the streaming kernels above.  A line of N
// cells is N / 32 independent loads instead of N / 32 loads one after the other, which is what a small grid needs
// ("not as much parallelism exposed as we could take advantage of"): at N = 256 a launch of the
// streaming kernels is 1024 warps that each wait for 8 tiles in turn.  Used for N <= 256 (and on request: NHP_FLAG_SECTIONS);
// from 512 cells on the streaming kernels already fill the machine and read each tile once without a barrier.
// ---------------------------------------------------------------------------------------------
constexpr uint32_t SX_D_CAP = 1u << 31;

template <bool UP, bool SOFT, int S = 0>
struct SummaryLoop {
    static __device__ __forceinline__ void run(const uint32_t *line, uint32_t &t, uint32_t &wp, uint32_t &d, uint32_t w, const uint4 &s0, const uint4 &s1)
    {
        constexpr int k = UP ? S : 31 - S;
        const uint32_t u = line[k];
        t = nhp_gate(nhp_arrive(t, wp, u), u);
        if (!SOFT) wp = w;
        if (SOFT) {
            const uint4 &q = (k < 16) ? s0 : s1;
            const uint32_t word = ((k >> 2) & 3) == 0 ? q.x : ((k >> 2) & 3) == 1 ? q.y : ((k >> 2) & 3) == 2 ? q.z : q.w;
            wp = nhp_soft_weight(w, word, k & 3);
            d += wp;
        }
        SummaryLoop<UP, SOFT, S + 1>::run(line, t, wp, d, w, s0, s1);
    }
};
template <bool UP, bool SOFT>
struct SummaryLoop<UP, SOFT, 32> {
    static __device__ __forceinline__ void run(const uint32_t *, uint32_t &, uint32_t &, uint32_t &, uint32_t, const uint4 &, const uint4 &) {}
};

template <bool SOFT>
__global__ void __launch_bounds__(512) straight_sect_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ Sline, const int16_t *__restrict__ B,
                                                            const uint32_t *__restrict__ xl_tab, const uint8_t *__restrict__ IJ,
                                                            const int16_t *__restrict__ tlist, int n_xslices, const uint32_t *__restrict__ lenq, uint32_t ct,
                                                            int log2_n, int is_forward, int fixed)
{
    extern __shared__ __align__(16) uint32_t smem[];
    const int n = 1 << log2_n, mx = n - 1, NT = n >> 5;
    const int xs = blockIdx.y, t = tlist[xs];
    const bool XS = xs < n_xslices;                                             // the list holds the slices with I = 0 first (block-uniform)
    const int lane = threadIdx.x & 31, T = threadIdx.x >> 5;                    // warp = tile T of the band
    const int X0 = blockIdx.x << 5;
    const bool up = (is_forward == ((IJ[t] >> 1) & 1));                         // eq (24)
    unsigned long long Vt = (unsigned long long)(V + ((size_t)t << (2 * log2_n)));
    asm volatile("" : "+l"(Vt));
    uint2 *sMD = (uint2 *)smem;                                                 // [NT][32]
    uint32_t *stage = smem + 2 * 32 * NT + T * XL_STAGE;                        // x-slices only
    const uint32_t w = SOFT ? lenq[t] << 4 : lenq[t];
    uint4 s0 = make_uint4(0, 0, 0, 0), s1 = s0;
    if (SOFT) {
        const uint8_t *Sl = Sline + ((size_t)t << (2 * log2_n)) + ((((size_t)blockIdx.x << (log2_n - 5)) + T) << 10) + 16 * lane;
        s0 = ld_nc16(Sl); s1 = ld_nc16(Sl + 512);
    }
    uint32_t u[32];
    uint32_t tw = 0;
    int bmine = 0;
    char *row = (char *)(stage + lane * XL_PITCH);
    const uint4 *offs4 = (const uint4 *)(stage + XL_DATA + 1);
    if (XS) {
        tw = xl_tab[((size_t)xs * NT + T) * 32 + lane];
        uint32_t nx[XL_ROWS];
        xl_tile_load<0>(nx, Vt, tw, T, X0, lane, log2_n);
        const int rows = (tw >> 8) & 63;
#pragma unroll
        for (int r = 0; r < XL_ROWS; r++)
            if (r < 32 || r < rows) stage[r * XL_PITCH + lane] = nx[r];
        stage[XL_DATA + 1 + lane] = (uint32_t)(((tw & 7) * XL_PITCH + lane) * 4);
        __syncwarp();
        xr_gather0(u, row, offs4);
    } else {
        bmine = B[(size_t)t * n + 32 * T + lane];
        const uint32_t row0 = (uint32_t)(32 * T) << log2_n, c0 = (uint32_t)(X0 + lane);
#pragma unroll
        for (int k = 0; k < 32; k++) {
            const int b = __shfl_sync(0xffffffffu, bmine, k);
            const uint32_t off = row0 + ((uint32_t)k << log2_n) + ((c0 + (uint32_t)b) & (uint32_t)mx);
            u[k] = *(const uint32_t *)(Vt + 4ull * off);
        }
    }
    // pass 1: (M, D) of this tile
    uint32_t lo = u[0];
#pragma unroll
    for (int k = 1; k + 1 < 32; k += 2) lo = __vimin3_u32(lo, u[k], u[k + 1]);
    const bool blocked_any = min(lo, u[31]) == 0u;
    {
        uint32_t tt = VI_INF, wp = 0u, d = 0u;
        if (up) SummaryLoop<true, SOFT>::run(u, tt, wp, d, w, s0, s1);
        else SummaryLoop<false, SOFT>::run(u, tt, wp, d, w, s0, s1);
        if (!SOFT) d = 32u * w;
        sMD[T * 32 + lane] = make_uint2(__viaddmin_u32(tt, wp, 0x7fffffffu), blocked_any ? SX_D_CAP : d);
    }
    __syncthreads();
    // ripple: the sections before this one, in travel order
    uint32_t c = VI_INF;
    if (up) { for (int p = 0; p < T; p++) { const uint2 md = sMD[p * 32 + lane]; c = __viaddmin_u32(c, md.y, md.x); } }
    else { for (int p = NT - 1; p > T; p--) { const uint2 md = sMD[p * 32 + lane]; c = __viaddmin_u32(c, md.y, md.x); } }
    // pass 2
    uint32_t cm = 0, wp = 0u;
    if (!fixed && tile_is_idle4(u, c)) { }
    else if (up) RelaxLoop<true, SOFT>::run(u, c, wp, w, ct, s0, s1, cm);
    else RelaxLoop<false, SOFT>::run(u, c, wp, w, ct, s0, s1, cm);
    if (fixed == 1) cm = 0xffffffffu;                       // NHP_FLAG_FIXED_WORK: every vertex goes back
    if (XS) {
        const uint32_t lines = __ballot_sync(0xffffffffu, cm != 0u);
        if (lines) {
            xr_scatter0(u, row, offs4, cm);
            __syncwarp();
            xl_stage_store(stage, Vt, tw, T, X0, lane, log2_n, lines);
        }
    } else if (__any_sync(0xffffffffu, cm != 0u)) {
        const uint32_t row0 = (uint32_t)(32 * T) << log2_n, c0 = (uint32_t)(X0 + lane);
#pragma unroll
        for (int k = 0; k < 32; k++) {
            const int b = __shfl_sync(0xffffffffu, bmine, k);
            const uint32_t off = row0 + ((uint32_t)k << log2_n) + ((c0 + (uint32_t)b) & (uint32_t)mx);
            if ((cm >> k) & 1u) st_global(Vt, off, u[k]);
        }
    }
}

}  // namespace

// SF or SB over the whole volume: one launch for the slices with I = 0 (tiles transposed through shared memory)
// and one for those with I = 1 (tiles in registers).  Returns the number of kernels launched (0 = not applicable).
int launch_straight_tile(nhp_planner *p, int m)
{
    const bool sparse = p->sparse_xp >= 0;
    const StartCurve sc{p->sparse_xp, p->sparse_yp, p->nt, p->d_beta, p->d_B};
    if (p->w.flags & NHP_FLAG_SIMPLE_KERNELS) return 0;
    const bool soft = p->S != nullptr;
    const int n = p->n, nt = p->nt;
    const int bands = n / 32, warps = bands < 4 ? bands : 4;
    ProfScope prof(p, m);
    const uint32_t *lenq = p->d_lenq + (size_t)m * nt;
    const int nx = p->n_xslices, ny = nt - nx;
    const dim3 gy(sparse ? 1 : bands / warps, ny);
    const int fwd = (m == M_SF);
    const int fixed = (p->w.flags & NHP_FLAG_FIXED_WORK) ? 1 : (p->w.flags & NHP_FLAG_NO_SHORTCUTS) ? 2 : 0;   // 1: no short cuts, store all; 2: no short cuts
    // Sections (one warp per tile, all tiles of a band at once): small grids, or on request; at most 16 tiles per line
    if (!sparse && bands <= 16 && !(p->w.flags & NHP_FLAG_NO_SECTIONS) && (n <= 256 || (p->w.flags & NHP_FLAG_SECTIONS))) {
        const size_t smx = sizeof(uint32_t) * (size_t)bands * (64 + XL_STAGE);
        ProfScope ps(p, 16);                                     // both slice groups in ONE launch (the block index tells which)
        if (soft) straight_sect_kernel<true><<<dim3(bands, nt), bands * 32, smx, p->stream>>>(p->V, p->S_line, p->d_B, p->d_xl_tab, p->d_IJ, p->d_tlist, nx, lenq, p->w.ct[m], p->log2_n, fwd, fixed);
        else straight_sect_kernel<false><<<dim3(bands, nt), bands * 32, smx, p->stream>>>(p->V, p->S_line, p->d_B, p->d_xl_tab, p->d_IJ, p->d_tlist, nx, lenq, p->w.ct[m], p->log2_n, fwd, fixed);
        return 1;
    }
    {
        const int xw = sparse ? 1 : bands < XL_WARPS_V ? bands : XL_WARPS_V;      // sparse: the one band that holds the line, one warp
        const size_t smem = sizeof(uint32_t) * (size_t)xw * XL_STAGE;
        const dim3 gx(sparse ? 1 : bands / xw, nx);
        ProfScope px(p, 14);
#define NHP_XL(SO, L2N) straight_xl_kernel<SO, L2N><<<gx, xw * 32, smem, p->stream>>>(p->V, p->S_line, p->d_xl_tab, p->d_IJ, p->d_tlist, lenq, p->w.ct[m], p->log2_n, fwd, fixed, sc)
        if (p->log2_n == 9) { if (soft) NHP_XL(true, 9); else NHP_XL(false, 9); }
        else if (p->log2_n == 10) { if (soft) NHP_XL(true, 10); else NHP_XL(false, 10); }
        else { if (soft) NHP_XL(true, 0); else NHP_XL(false, 0); }
#undef NHP_XL
    }
    {
        ProfScope py(p, 15);
        if (soft) straight_rows_kernel<true><<<gy, warps * 32, 0, p->stream>>>(p->V, p->S_line, p->d_B, p->d_IJ, p->d_tlist + nx, lenq, p->w.ct[m], p->log2_n, fwd, fixed, sc);
        else straight_rows_kernel<false><<<gy, warps * 32, 0, p->stream>>>(p->V, nullptr, p->d_B, p->d_IJ, p->d_tlist + nx, lenq, p->w.ct[m], p->log2_n, fwd, fixed, sc);
    }
    return 2;
}

int set_softlayout_attributes();               // softlayout.cu

// Function attributes are per device: set for the handle's device (current here) at creation.
int set_kernel_attributes(nhp_planner *p)
{
    (void)p;
    const int sect_smem = 4 * 16 * (64 + XL_STAGE);
    if (cudaFuncSetAttribute(straight_sect_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sect_smem) != cudaSuccess ||
        cudaFuncSetAttribute(straight_sect_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, sect_smem) != cudaSuccess)
        return NHP_E_CUDA;
    return set_softlayout_attributes();
}
