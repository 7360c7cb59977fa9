// Straight sweeps SF / SB, B200 version.
// PAPER.md:271-302 (section V.C, eqs (19)-(24): the discretised lines of one Theta slice), l.294 (direction by
// J), l.356 (one lap, started at the wall), Insert 5 l.946-949 (loop body), l.366-370 (the coalescing problem the
// paper solves with transposed slices and that is solved here by staging tiles in shared memory).
//
// One WARP owns a band of 32 neighbouring lines x' in [X0, X0+32) of one slice and walks along them in tiles of
// 32 sweep steps, carrying the travelling value of its 32 lines in registers (thread = line):
//   * slices with I = 1 (straight_rows_kernel): step = j, i = (x' + B(j)) & mask: every step is one (misaligned)
//     128-byte row segment in which lane l's word already is line l's vertex; tiles live in registers;
//   * slices with I = 0 (straight_xrows_kernel): step = i, j = (x' + B(i)) & mask, eq (23): the lines run along the
//     memory-fast axis; tiles are parallelograms of the slice, staged row-major in shared memory by 16-byte
//     cp.async, XR_NBUF - 1 tiles ahead, and read line-wise from there.
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
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void *gptr)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_addr), "l"(gptr) : "memory");
}

__device__ __forceinline__ uint4 ld_nc16(const uint8_t *p)
{
    uint4 q;
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(q.x), "=r"(q.y), "=r"(q.z), "=r"(q.w) : "l"(p));
    return q;
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
// vertices to 2^32 - 1 and is >= 2^30 for unreached ones): the relaxation cannot change anything.
__device__ __forceinline__ bool tile_is_idle(const uint32_t (&u)[32], uint32_t t)
{
    uint32_t lowest = 0xffffffffu;
#pragma unroll
    for (int k = 0; k < 32; k++) lowest = __viaddmin_u32(u[k], 0xffffffffu, lowest);
    return __all_sync(0xffffffffu, t >= VI_INF && lowest >= VI_INF - 1u);
}

// ---------------------------------------------------------------------------------------------
// Slices with I = 0 (|tan| <= 1, eq (19)): the sweep step is the COLUMN i and line x' sits at row
// (x' + B(i)) & mask, eq (23): the lines run along the memory-fast axis, so "thread = line" needs a transposition
// (the problem the paper solves by storing these slices transposed, l.366-370).  Here a warp owns a band of 32
// neighbouring lines and walks along it in tiles of 32 columns.  A tile is a parallelogram of the slice, rows
// r_min .. r_min + 31 + span (span = |B(i0 + 31) - B(i0)| <= 31).  It is staged ROW-MAJOR in shared memory by 16-byte
// cp.async: 8 lanes fetch the 8 aligned chunks of one row segment, four rows per warp instruction, only the chunks
// the parallelogram touches (a 4-byte cp.async costs the LSU as much per instruction as a 16-byte one and moved the
// same tile with 64 instructions instead of <= 16: the kernel was bound by exactly that, profiles/r01_tile_kernels.md).
// The line of thread l then reads column k at row l + delta_k, delta_k = B(i0 + k) - B_min: rows are 36 words apart,
// so the 32 lanes fall on 8 banks (4-way conflict, 4 cycles per warp load; the 16-byte alignment of the rows rules
// out an odd stride).  Improved values go back into the staged tile and from there, row by row, to the volume.
// ---------------------------------------------------------------------------------------------
constexpr int XR_RS = 36;                                  // words per staged row segment (32 + 4: rows stay 16-byte aligned)
constexpr int XR_ROWS = 35;                                // staged rows: 32 lines + 3 (slope inside a chunk) + 1, see xr_stage_load
#ifndef XR_NBUF_V
#define XR_NBUF_V 3
#endif
#ifndef XR_WARPS_V
#define XR_WARPS_V 1
#endif
constexpr int XR_NBUF = XR_NBUF_V;                                 // tiles in flight per warp
constexpr int XR_TILE_WORDS = XR_ROWS * XR_RS + 32;        // + byte offset delta_k * XR_RS * 4 of every column

// gather / scatter the 32 columns of this thread's line from / to the staged tile.  `row` points at (row l, column 0),
// offs4 at the table of byte offsets delta_k * 144 (warp-uniform, read four at a time)
__device__ __forceinline__ void xr_gather(uint32_t (&u)[32], const char *row, const uint4 *offs4)
{
#pragma unroll
    for (int q = 0; q < 8; q++) {
        const uint4 o = offs4[q];
        u[4 * q + 0] = *(const uint32_t *)(row + o.x + 16 * q);
        u[4 * q + 1] = *(const uint32_t *)(row + o.y + 16 * q + 4);
        u[4 * q + 2] = *(const uint32_t *)(row + o.z + 16 * q + 8);
        u[4 * q + 3] = *(const uint32_t *)(row + o.w + 16 * q + 12);
    }
}
__device__ __forceinline__ void xr_scatter(const uint32_t (&u)[32], char *row, const uint4 *offs4, uint32_t cm)
{
#pragma unroll
    for (int q = 0; q < 8; q++) {
        const uint4 o = offs4[q];
        if ((cm >> (4 * q + 0)) & 1u) *(uint32_t *)(row + o.x + 16 * q) = u[4 * q + 0];
        if ((cm >> (4 * q + 1)) & 1u) *(uint32_t *)(row + o.y + 16 * q + 4) = u[4 * q + 1];
        if ((cm >> (4 * q + 2)) & 1u) *(uint32_t *)(row + o.z + 16 * q + 8) = u[4 * q + 2];
        if ((cm >> (4 * q + 3)) & 1u) *(uint32_t *)(row + o.w + 16 * q + 12) = u[4 * q + 3];
    }
}

// cp.async of tile T of the band [X0, X0 + 32) into the stage at shared byte address `stage` (generic pointer `sp`)
template <bool SOFT>
__device__ __forceinline__ void xr_stage_load(uint32_t stage, uint32_t *sp, unsigned long long Vt, const uint8_t *__restrict__ Sl,
                                              const int16_t *__restrict__ Bt, int T, int X0, int lane, int log2_n)
{
    const int mx = (1 << log2_n) - 1;
    const int bmine = Bt[32 * T + lane];
    // B(i) is monotone in i, so its extremes over the tile sit in lanes 0 and 31
    const int b0 = __shfl_sync(0xffffffffu, bmine, 0), b31 = __shfl_sync(0xffffffffu, bmine, 31);
    const int bmin = min(b0, b31), nrows = 32 + abs(b31 - b0);
    const int delta = bmine - bmin;                            // line l meets column `lane` in row l + delta of the parallelogram
    // The stage is SHEARED chunk by chunk: the 16-byte chunk (row q, columns 4c .. 4c+3) goes to stage row q - dlo(c),
    // dlo(c) = the smallest delta of its four columns.  The parallelogram (up to 63 rows) then fits 32 + 3 stage rows,
    // and line l finds column k in stage row l + delta_k - dlo(k / 4), a per-column offset the relax loop reads from a table.
    const int my4 = lane & ~3;
    const int dl0 = __shfl_sync(0xffffffffu, delta, my4), dl3 = __shfl_sync(0xffffffffu, delta, my4 + 3);
    sp[XR_ROWS * XR_RS + lane] = (uint32_t)((delta - min(dl0, dl3)) * (XR_RS * 4));
    // chunk c of a row; the parallelogram touches it in rows [dlo, dhi + 31]
    const int c = lane & 7, qs = lane >> 3;
    const int d0 = __shfl_sync(0xffffffffu, delta, 4 * c), d3 = __shfl_sync(0xffffffffu, delta, 4 * c + 3);
    const int dlo = min(d0, d3), dhi = max(d0, d3) + 31;
    const int rmin = X0 + bmin;
    const uint32_t col = (uint32_t)(32 * T + 4 * c);
    uint32_t sa = stage + 4u * (uint32_t)((qs - dlo) * XR_RS + 4 * c);
    for (int q = qs; q < nrows; q += 4) {                      // warp-uniform trip count: one instruction = four rows of the slice
        if (q >= dlo && q <= dhi) {
            const uint32_t off = ((uint32_t)((rmin + q) & mx) << log2_n) + col;
            cp_async16(sa, (const void *)(Vt + 4ull * off));
        }
        sa += 4u * 4u * XR_RS;
    }
    if (SOFT) {
        // S_line[Theta][x'][y']: this lane's line, steps 32 T .. 32 T + 31 = 32 contiguous bytes ([half][lane] uint4)
        const uint8_t *g = Sl + (((size_t)(X0 + lane)) << log2_n) + 32 * T;
        const uint32_t ss = stage + 4u * (uint32_t)XR_TILE_WORDS + 16u * (uint32_t)lane;
        cp_async16(ss, g);
        cp_async16(ss + 512u, g + 16);
    }
}

// rows of the staged tile back to the volume: element (row q, column lane) belongs to line q - delta; `lines` = the
// lines of the band with an improved value
__device__ __forceinline__ void xr_stage_store(const uint32_t *sp, unsigned long long Vt, const int16_t *__restrict__ Bt, int T, int X0,
                                               int lane, int log2_n, uint32_t lines)
{
    const int mx = (1 << log2_n) - 1;
    const int bmine = Bt[32 * T + lane];
    const int b0 = __shfl_sync(0xffffffffu, bmine, 0), b31 = __shfl_sync(0xffffffffu, bmine, 31);
    const int bmin = min(b0, b31), nrows = 32 + abs(b31 - b0);
    const int delta = bmine - bmin;
    // bit q of `want`: this column's vertex in row q sits on a line that improved
    const unsigned long long want = (unsigned long long)lines << delta;
    const int my4 = lane & ~3;
    const int dl0 = __shfl_sync(0xffffffffu, delta, my4), dl3 = __shfl_sync(0xffffffffu, delta, my4 + 3);
    const uint32_t *s = sp + lane - min(dl0, dl3) * XR_RS;   // row q of the slice is stage row q - dlo(lane / 4)
    // only the rows between the first and the last improved line; element offsets step by one row, wrapped on the torus
    const int q0 = __ffs(lines) - 1, q1 = 32 - __clz(lines) + (nrows - 32);
    const uint32_t smask = (1u << (2 * log2_n)) - 1u, rstep = 1u << log2_n;
    uint32_t off = ((((uint32_t)(X0 + bmin + q0)) << log2_n) & smask) + (uint32_t)(32 * T + lane);
    uint32_t wlo = (uint32_t)(want >> q0), whi = (uint32_t)((want >> q0) >> 32);
    s += q0 * XR_RS;
    for (int q = q0; q < q1; q += 4) {                        // warp-uniform bounds
#pragma unroll
        for (int e = 0; e < 4; e++) {
            if ((wlo >> e) & 1u) st_global(Vt, off, s[e * XR_RS]);
            off = (off + rstep) & smask;
        }
        wlo = __funnelshift_r(wlo, whi, 4);
        whi >>= 4;
        s += 4 * XR_RS;
    }
}

template <bool SOFT>
__device__ __forceinline__ void xr_band_sweep(uint32_t *__restrict__ Vslice, const uint8_t *__restrict__ Sl, const int16_t *__restrict__ Bt,
                                              uint32_t *buf, int X0, int lane, int log2_n, uint32_t w, uint32_t ct, bool up, int fixed)
{
    constexpr int SW = XR_TILE_WORDS + (SOFT ? 256 : 0);
    const int NT = 1 << (log2_n - 5);
    unsigned long long Vt = (unsigned long long)Vslice;
    asm volatile("" : "+l"(Vt));
    const uint32_t sbuf = (uint32_t)__cvta_generic_to_shared(buf);
    for (int s = 0; s < XR_NBUF - 1; s++) {
        if (s < NT) xr_stage_load<SOFT>(sbuf + 4u * (uint32_t)(s * SW), buf + s * SW, Vt, Sl, Bt, up ? s : NT - 1 - s, X0, lane, log2_n);
        cp_async_commit();
    }
    uint32_t t = VI_INF, wp = SOFT ? 0u : w;          // nothing arrives at the wall cell the line starts from
    int b = 0, bn = XR_NBUF - 1;                      // buffer of tile s, buffer of tile s + NBUF - 1
#pragma unroll 1
    for (int s = 0; s < NT; s++) {
        cp_async_wait<XR_NBUF - 2>();
        __syncwarp();
        {   // prefetch tile s + NBUF - 1 into the buffer tile s - 1 has just left
            const int sn = s + XR_NBUF - 1;
            if (sn < NT) xr_stage_load<SOFT>(sbuf + 4u * (uint32_t)(bn * SW), buf + bn * SW, Vt, Sl, Bt, up ? sn : NT - 1 - sn, X0, lane, log2_n);
            cp_async_commit();
        }
        uint32_t *tile = buf + b * SW;
        char *row = (char *)(tile + lane * XR_RS);
        const uint4 *offs4 = (const uint4 *)(tile + XR_ROWS * XR_RS);
        uint32_t u[32];
        xr_gather(u, row, offs4);
        uint4 s0 = make_uint4(0, 0, 0, 0), s1 = s0;
        if (SOFT) {
            const uint4 *sl = (const uint4 *)(tile + XR_TILE_WORDS);
            s0 = sl[lane]; s1 = sl[32 + lane];
        }
        uint32_t cm = 0;
        if (!fixed && tile_is_idle(u, t)) { }
        else if (up) RelaxLoop<true, SOFT>::run(u, t, wp, w, ct, s0, s1, cm);
        else RelaxLoop<false, SOFT>::run(u, t, wp, w, ct, s0, s1, cm);
        if (fixed) cm = 0xffffffffu;                       // NHP_FLAG_FIXED_WORK: every vertex goes back
        const uint32_t lines = __ballot_sync(0xffffffffu, cm != 0u);
        if (lines) {
            xr_scatter(u, row, offs4, cm);
            __syncwarp();
            xr_stage_store(tile, Vt, Bt, up ? s : NT - 1 - s, X0, lane, log2_n, lines);
        }
        b = (b + 1 == XR_NBUF) ? 0 : b + 1;
        bn = (bn + 1 == XR_NBUF) ? 0 : bn + 1;
    }
}

template <bool SOFT>
__global__ void __launch_bounds__(128) straight_xrows_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ Sline,
                                                             const int16_t *__restrict__ B, const uint8_t *__restrict__ IJ,
                                                             const int16_t *__restrict__ tlist,
                                                             const uint32_t *__restrict__ lenq, uint32_t ct, int log2_n, int is_forward, int fixed)
{
    extern __shared__ __align__(16) uint32_t smem[];
    constexpr int SW = XR_TILE_WORDS + (SOFT ? 256 : 0);
    const int n = 1 << log2_n, t = tlist[blockIdx.y];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int X0 = (blockIdx.x * (blockDim.x >> 5) + warp) << 5;
    const int jpos = (IJ[t] >> 1) & 1;
    const bool up = (is_forward == jpos);                                       // eq (24)
    const int16_t *Bt = B + (size_t)t * n;
    uint32_t *Vt = V + ((size_t)t << (2 * log2_n));
    const uint8_t *Sl = SOFT ? Sline + ((size_t)t << (2 * log2_n)) : nullptr;
    uint32_t *buf = smem + warp * (XR_NBUF * SW);
    const uint32_t w = SOFT ? lenq[t] << 4 : lenq[t];
    xr_band_sweep<SOFT>(Vt, Sl, Bt, buf, X0, lane, log2_n, w, ct, up, fixed);
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
                                                            const uint32_t *__restrict__ lenq, uint32_t ct, int log2_n, int is_forward, int fixed)
{
    const int n = 1 << log2_n, mx = n - 1, t = tlist[blockIdx.y];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int X0 = (blockIdx.x * (blockDim.x >> 5) + warp) << 5;
    const int jpos = (IJ[t] >> 1) & 1;
    const bool up = (is_forward == jpos);                                       // eq (24)
    const int16_t *Bt = B + (size_t)t * n;
    unsigned long long Vt = (unsigned long long)(V + ((size_t)t << (2 * log2_n)));
    asm volatile("" : "+l"(Vt));
    const uint8_t *Sl = SOFT ? Sline + ((size_t)t << (2 * log2_n)) + ((size_t)(X0 + lane) << log2_n) : nullptr;
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
        if (SOFT) { s0 = ld_nc16(Sl + 32 * T); s1 = ld_nc16(Sl + 32 * T + 16); }
        uint32_t cm = 0;
        if (!fixed && tile_is_idle(u, tv)) { }
        else if (up) RelaxLoop<true, SOFT>::run(u, tv, wp, w, ct, s0, s1, cm);
        else RelaxLoop<false, SOFT>::run(u, tv, wp, w, ct, s0, s1, cm);
        if (fixed) cm = 0xffffffffu;                       // NHP_FLAG_FIXED_WORK: every vertex goes back
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

}  // namespace

// SF or SB over the whole volume: one launch for the slices with I = 0 (tiles transposed through shared memory)
// and one for those with I = 1 (tiles in registers).  Returns the number of kernels launched (0 = not applicable).
int launch_straight_tile(nhp_planner *p, int m)
{
    if (p->w.flags & NHP_FLAG_SIMPLE_KERNELS) return 0;
    const bool soft = p->S != nullptr;
    const int n = p->n, nt = p->nt;
    const int bands = n / 32, warps = bands < 4 ? bands : 4, xwarps = bands < XR_WARPS_V ? bands : XR_WARPS_V;
    const int sw = XR_TILE_WORDS + (soft ? 256 : 0);
    const size_t smem = sizeof(uint32_t) * (size_t)xwarps * XR_NBUF * sw;
    ProfScope prof(p, m);
    const uint32_t *lenq = p->d_lenq + (size_t)m * nt;
    const int nx = p->n_xslices, ny = nt - nx;
    const dim3 gx(bands / xwarps, nx), gy(bands / warps, ny);
    const int fwd = (m == M_SF);
    const int fixed = (p->w.flags & NHP_FLAG_FIXED_WORK) ? 1 : 0;
    if (soft) {
        { ProfScope px(p, 14); straight_xrows_kernel<true><<<gx, xwarps * 32, smem, p->stream>>>(p->V, p->S_line, p->d_B, p->d_IJ, p->d_tlist, lenq, p->w.ct[m], p->log2_n, fwd, fixed); }
        { ProfScope py(p, 15); straight_rows_kernel<true><<<gy, warps * 32, 0, p->stream>>>(p->V, p->S_line, p->d_B, p->d_IJ, p->d_tlist + nx, lenq, p->w.ct[m], p->log2_n, fwd, fixed); }
    } else {
        { ProfScope px(p, 14); straight_xrows_kernel<false><<<gx, xwarps * 32, smem, p->stream>>>(p->V, nullptr, p->d_B, p->d_IJ, p->d_tlist, lenq, p->w.ct[m], p->log2_n, fwd, fixed); }
        { ProfScope py(p, 15); straight_rows_kernel<false><<<gy, warps * 32, 0, p->stream>>>(p->V, nullptr, p->d_B, p->d_IJ, p->d_tlist + nx, lenq, p->w.ct[m], p->log2_n, fwd, fixed); }
    }
    return 2;
}

int set_softlayout_attributes();               // softlayout.cu

// Function attributes are per device: set for the handle's device (current here) at creation.
int set_kernel_attributes(nhp_planner *p)
{
    (void)p;
    if (cudaFuncSetAttribute(straight_xrows_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * XR_NBUF * XR_TILE_WORDS * 4) != cudaSuccess ||
        cudaFuncSetAttribute(straight_xrows_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * XR_NBUF * (XR_TILE_WORDS + 256) * 4) != cudaSuccess)
        return NHP_E_CUDA;
    return set_softlayout_attributes();
}
