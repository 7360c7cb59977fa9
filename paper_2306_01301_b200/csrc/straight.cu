// Straight sweeps SF / SB, B200 version.
// PAPER.md:271-302 (section V.C, eqs (19)-(24): the discretised lines of one Theta slice), l.294 (direction by
// J), l.356 (one lap, started at the wall), Insert 5 l.946-949 (loop body), l.366-370 (the coalescing problem the
// paper solves with transposed slices and that is solved here by staging tiles in shared memory).
//
// One WARP owns a band of 32 neighbouring lines x' in [X0, X0+32) of one slice and walks along them in tiles of
// 32 sweep steps, carrying the arriving value v of its 32 lines in registers (thread = line).  Tiles are brought
// into shared memory by cp.async, ST_NBUF - 1 tiles ahead of the one being relaxed, so that the dependent chain
// of a line never waits for HBM.  In shared memory element (line l, step k) of a tile sits at word l*33 + k:
//   * slices with I = 0 (|tan| <= 1, eq (19)): step = i, j = (x' + B(i)) & mask, eq (23).  The tile is a
//     parallelogram of the slice: rows r0 .. r0+31+span, 128-byte row segments, each lane (= column i) copying
//     the 32 rows that belong to its column; the transposition to "thread = line" happens in the shared-memory
//     addressing, both directions conflict-free (bank = l + k).
//   * slices with I = 1: step = j, i = (x' + B(j)) & mask: every step is one (misaligned) 128-byte row segment.
// A tile is written back (again as row segments) only if a value in it improved.
#include "nhp_internal.cuh"

namespace {

constexpr int ST_NBUF = 3;                 // tiles in flight per warp (one being relaxed, two arriving)
constexpr int ST_STRIDE = 33;              // words per line in a tile (padding -> conflict-free both ways)
constexpr int ST_TILE_WORDS = 32 * ST_STRIDE;

// Global addresses are formed as (opaque 64-bit slice base) + 4 * (32-bit element offset): one IMAD.WIDE.  The base
// is made opaque once per warp so that the compiler keeps it in a register pair instead of re-deriving it from
// the kernel parameters at every row.
__device__ __forceinline__ void cp_async4(uint32_t smem_addr, unsigned long long vbase, uint32_t off)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(smem_addr), "l"(vbase + 4ull * off) : "memory");
}
__device__ __forceinline__ void st_global(unsigned long long vbase, uint32_t off, uint32_t val)
{
    asm volatile("st.global.u32 [%0], %1;\n" ::"l"(vbase + 4ull * off), "r"(val) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// Geometry of one tile of a band, as the load and the store phase need it (recomputed, never kept: 3 registers).
struct TileGeo {
    int delta;                 // class X: first row of this lane's column inside the parallelogram
    int row0, rdir, nrows;     // class X: rows (row0 + rdir q) & mask, q < nrows <= 64
    int bmine;                 // B(32 T + lane): class Y broadcasts it row by row
};

template <bool XCLASS>
__device__ __forceinline__ TileGeo tile_geometry(const int16_t *__restrict__ Bt, int T, int X0, int lane, bool pos)
{
    TileGeo g;
    g.bmine = Bt[32 * T + lane];
    g.delta = 0; g.row0 = 0; g.rdir = 1; g.nrows = 32;
    if (XCLASS) {
        // B(i) is monotone in i, so its extremes over the tile sit in lanes 0 and 31
        const int b0 = __shfl_sync(0xffffffffu, g.bmine, 0), b31 = __shfl_sync(0xffffffffu, g.bmine, 31);
        const int bmin = min(b0, b31), bmax = max(b0, b31);
        // rows are numbered so that delta is non-increasing in the lane index (conflict-free staging, see top)
        g.delta = pos ? bmax - g.bmine : g.bmine - bmin;
        g.row0 = pos ? X0 + bmax + 31 : X0 + bmin;
        g.rdir = pos ? -1 : 1;
        g.nrows = 32 + bmax - bmin;
    }
    return g;
}

// cp.async of tile T into `tile` (shared-memory byte address of the warp's buffer).  The row loops are unrolled
// by 8 only: the whole kernel has to stay inside the instruction cache (a fully unrolled version ran at
// "no instruction" stalls of 3-7 per issue, profiles/r01_tile_kernels.md).
template <bool XCLASS>
__device__ __forceinline__ void tile_load(uint32_t tile, unsigned long long Vt, const int16_t *__restrict__ Bt, int T,
                                          int X0, int lane, int log2_n, bool pos)
{
    const int mx = (1 << log2_n) - 1;
    const TileGeo g = tile_geometry<XCLASS>(Bt, T, X0, lane, pos);
    if (XCLASS) {
        // lane = column i = 32 T + lane; row q of the parallelogram goes to line (q - delta) of the tile
        uint32_t sa = tile + 4u * (uint32_t)(lane - g.delta * ST_STRIDE);
        unsigned long long act = 0xffffffffull << g.delta;                      // bit q: my column owns row q
        // element offset inside the slice; "& smask" wraps the row index (the slice is a torus)
        const uint32_t smask = (1u << (2 * log2_n)) - 1u, rstep = (uint32_t)(g.rdir << log2_n);
        uint32_t off = (((uint32_t)g.row0 << log2_n) + (uint32_t)(32 * T + lane)) & smask;
        for (int q0 = 0; q0 < g.nrows; q0 += 8) {                                // warp-uniform trip count
#pragma unroll
            for (int qq = 0; qq < 8; qq++) {
                if (((uint32_t)act >> qq) & 1u) cp_async4(sa + 4u * (uint32_t)(qq * ST_STRIDE), Vt, off);
                off = (off + rstep) & smask;
            }
            act >>= 8;
            sa += 4u * 8u * ST_STRIDE;
        }
    } else {
        // step k = row j = 32 T + k; lane = line: column (X0 + B(j) + lane) & mask
        const uint32_t sa = tile + 4u * (uint32_t)(lane * ST_STRIDE);
        const uint32_t c0 = (uint32_t)(X0 + lane), n = 1u << log2_n;
        uint32_t rowoff = (uint32_t)(32 * T) << log2_n;
#pragma unroll 8
        for (int k = 0; k < 32; k++) {
            const int b = __shfl_sync(0xffffffffu, g.bmine, k);
            cp_async4(sa + 4u * (uint32_t)k, Vt, rowoff + ((c0 + (uint32_t)b) & (uint32_t)mx));
            rowoff += n;
        }
    }
}

// write tile T back; cm = this thread's (= line's) mask of improved steps
template <bool XCLASS>
__device__ __forceinline__ void tile_store(const uint32_t *tile, unsigned long long Vt, const int16_t *__restrict__ Bt, int T,
                                           int X0, int lane, int log2_n, bool pos, uint32_t cm)
{
    const int mx = (1 << log2_n) - 1;
    const TileGeo g = tile_geometry<XCLASS>(Bt, T, X0, lane, pos);
    if (XCLASS) {
        const uint32_t lines = __ballot_sync(0xffffffffu, cm != 0u);             // lines with an improved value
        const uint32_t *sb = tile + (lane - g.delta * ST_STRIDE);
        unsigned long long want = (unsigned long long)lines << g.delta;          // rows of my column on those lines
        const uint32_t smask = (1u << (2 * log2_n)) - 1u, rstep = (uint32_t)(g.rdir << log2_n);
        uint32_t off = (((uint32_t)g.row0 << log2_n) + (uint32_t)(32 * T + lane)) & smask;
        for (int q0 = 0; q0 < g.nrows; q0 += 8) {
#pragma unroll
            for (int qq = 0; qq < 8; qq++) {
                if (((uint32_t)want >> qq) & 1u) st_global(Vt, off, sb[qq * ST_STRIDE]);
                off = (off + rstep) & smask;
            }
            want >>= 8;
            sb += 8 * ST_STRIDE;
        }
    } else {
        const uint32_t *sb = tile + lane * ST_STRIDE;
        const uint32_t c0 = (uint32_t)(X0 + lane), n = 1u << log2_n;
        uint32_t rowoff = (uint32_t)(32 * T) << log2_n;
#pragma unroll 8
        for (int k = 0; k < 32; k++) {
            const int b = __shfl_sync(0xffffffffu, g.bmine, k);
            if ((cm >> k) & 1u) st_global(Vt, rowoff + ((c0 + (uint32_t)b) & (uint32_t)mx), sb[k]);
            rowoff += n;
        }
    }
}

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

// Relax the 32 steps of a tile for this thread's line (Insert 5, internal encoding):
//   V[i] = min(v, u);  v = min(v, u + ct) + (blocked ? infinity : w)          (nhp_chain_step)
// Soft: w = (len_q * S) >> 4 per vertex, S from the line-major copy of the soft volume (sl: this line's 32 bytes).
template <bool UP, bool SOFT, int S = 0>
struct RelaxLoop {
    static __device__ __forceinline__ void run(uint32_t *line, uint32_t &v, uint32_t w, uint32_t ct, const uint4 &s0, const uint4 &s1,
                                               uint32_t &cm)
    {
        constexpr int k = UP ? S : 31 - S;
        const uint32_t u = line[k];
        if (v < u) { line[k] = v; cm |= 1u << k; }
        uint32_t wk = w;
        if (SOFT) {
            const uint4 &q = (k < 16) ? s0 : s1;
            const uint32_t word = ((k >> 2) & 3) == 0 ? q.x : ((k >> 2) & 3) == 1 ? q.y : ((k >> 2) & 3) == 2 ? q.z : q.w;
            wk = nhp_soft_weight(w, word, k & 3);
        }
        v = nhp_chain_step(v, u, wk, ct);
        RelaxLoop<UP, SOFT, S + 1>::run(line, v, w, ct, s0, s1, cm);
    }
};
template <bool UP, bool SOFT>
struct RelaxLoop<UP, SOFT, 32> {
    static __device__ __forceinline__ void run(uint32_t *, uint32_t &, uint32_t, uint32_t, const uint4 &, const uint4 &, uint32_t &) {}
};

template <bool UP, bool SOFT>
__device__ __forceinline__ uint32_t tile_relax(uint32_t *line, const uint4 *sl, int lane, uint32_t &v, uint32_t w, uint32_t ct)
{
    uint32_t cm = 0;
    uint4 s0 = make_uint4(0, 0, 0, 0), s1 = s0;
    if (SOFT) { s0 = sl[lane]; s1 = sl[32 + lane]; }
    RelaxLoop<UP, SOFT>::run(line, v, w, ct, s0, s1, cm);
    return cm;
}

// One pipeline stage of a warp = the V tile and, with soft costs, the 32 x 32 bytes of S behind it ([half][lane] uint4).
template <bool XCLASS, bool SOFT>
__device__ __forceinline__ void stage_load(uint32_t stage, unsigned long long Vt, const uint8_t *__restrict__ Sl, const int16_t *__restrict__ Bt,
                                           int T, int X0, int lane, int log2_n, bool pos)
{
    tile_load<XCLASS>(stage, Vt, Bt, T, X0, lane, log2_n, pos);
    if (SOFT) {
        // S_line[Theta][x'][y']: this lane's line, steps 32 T .. 32 T + 31 = 32 contiguous bytes.  In class-X tiles
        // with K > 0 the rows are numbered downwards (tile_geometry), so thread `lane` owns line X0 + 31 - lane.
        const int xl = (XCLASS && pos) ? 31 - lane : lane;
        const uint8_t *g = Sl + (((size_t)(X0 + xl)) << log2_n) + 32 * T;
        const uint32_t sa = stage + 4u * (uint32_t)ST_TILE_WORDS + 16u * (uint32_t)lane;
        cp_async16(sa, g);
        cp_async16(sa + 512u, g + 16);
    }
}

template <bool XCLASS, bool SOFT>
__device__ __forceinline__ void band_sweep(uint32_t *__restrict__ Vslice, const uint8_t *__restrict__ Sl, const int16_t *__restrict__ Bt,
                                           uint32_t *buf, int X0, int lane, int log2_n, uint32_t w, uint32_t ct, bool pos, bool up)
{
    constexpr int SW = ST_TILE_WORDS + (SOFT ? 256 : 0);
    const int NT = 1 << (log2_n - 5);
    unsigned long long Vt = (unsigned long long)Vslice;
    asm volatile("" : "+l"(Vt));
    const uint32_t sbuf = (uint32_t)__cvta_generic_to_shared(buf);
    for (int s = 0; s < ST_NBUF - 1; s++) {
        if (s < NT) stage_load<XCLASS, SOFT>(sbuf + 4u * (uint32_t)(s * SW), Vt, Sl, Bt, up ? s : NT - 1 - s, X0, lane, log2_n, pos);
        cp_async_commit();
    }
    uint32_t v = VI_INF;
    int b = 0, bn = ST_NBUF - 1;                      // buffer of tile s, buffer of tile s + NBUF - 1
#pragma unroll 1
    for (int s = 0; s < NT; s++) {
        cp_async_wait<ST_NBUF - 2>();
        __syncwarp();
        {   // prefetch tile s + NBUF - 1 into the buffer tile s - 1 has just left
            const int sn = s + ST_NBUF - 1;
            if (sn < NT) stage_load<XCLASS, SOFT>(sbuf + 4u * (uint32_t)(bn * SW), Vt, Sl, Bt, up ? sn : NT - 1 - sn, X0, lane, log2_n, pos);
            cp_async_commit();
        }
        uint32_t *tile = buf + b * SW;
        const uint4 *sl = (const uint4 *)(tile + ST_TILE_WORDS);
        const uint32_t cm = up ? tile_relax<true, SOFT>(tile + lane * ST_STRIDE, sl, lane, v, w, ct)
                               : tile_relax<false, SOFT>(tile + lane * ST_STRIDE, sl, lane, v, w, ct);
        if (__any_sync(0xffffffffu, cm != 0u)) {
            __syncwarp();
            tile_store<XCLASS>(tile, Vt, Bt, up ? s : NT - 1 - s, X0, lane, log2_n, pos, cm);
        }
        b = (b + 1 == ST_NBUF) ? 0 : b + 1;
        bn = (bn + 1 == ST_NBUF) ? 0 : bn + 1;
    }
}

template <bool SOFT>
__global__ void __launch_bounds__(128) straight_tile_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ Sline,
                                                            const int16_t *__restrict__ B, const uint8_t *__restrict__ IJ,
                                                            const int16_t *__restrict__ tlist,
                                                            const uint32_t *__restrict__ lenq, uint32_t ct, int log2_n, int is_forward)
{
    extern __shared__ __align__(16) uint32_t smem[];
    constexpr int SW = ST_TILE_WORDS + (SOFT ? 256 : 0);
    const int n = 1 << log2_n, t = tlist[blockIdx.y];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int X0 = (blockIdx.x * (blockDim.x >> 5) + warp) << 5;
    const int I = IJ[t] & 1, jpos = (IJ[t] >> 1) & 1;
    const bool up = (is_forward == jpos);                                       // eq (24)
    const int16_t *Bt = B + (size_t)t * n;
    const bool pos = Bt[n - 1] >= 0;                                            // sign of K(Theta), eq (20)
    uint32_t *Vt = V + ((size_t)t << (2 * log2_n));
    const uint8_t *Sl = SOFT ? Sline + ((size_t)t << (2 * log2_n)) : nullptr;
    uint32_t *buf = smem + warp * (ST_NBUF * SW);
    const uint32_t w = SOFT ? lenq[t] << 4 : lenq[t];
    if (I == 0) band_sweep<true, SOFT>(Vt, Sl, Bt, buf, X0, lane, log2_n, w, ct, pos, up);
    else band_sweep<false, SOFT>(Vt, Sl, Bt, buf, X0, lane, log2_n, w, ct, pos, up);
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
__global__ void __launch_bounds__(128, 8) straight_rows_kernel(uint32_t *__restrict__ V, const uint8_t *__restrict__ Sline,
                                                            const int16_t *__restrict__ B, const uint8_t *__restrict__ IJ,
                                                            const int16_t *__restrict__ tlist,
                                                            const uint32_t *__restrict__ lenq, uint32_t ct, int log2_n, int is_forward)
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
    uint32_t v = VI_INF;
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
        if (up) RelaxLoop<true, SOFT>::run(u, v, w, ct, s0, s1, cm);
        else RelaxLoop<false, SOFT>::run(u, v, w, ct, s0, s1, cm);
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
    const int bands = n / 32, warps = bands < 4 ? bands : 4;
    const int sw = ST_TILE_WORDS + (soft ? 256 : 0);
    const size_t smem = sizeof(uint32_t) * (size_t)warps * ST_NBUF * sw;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(straight_tile_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * ST_NBUF * ST_TILE_WORDS * 4);
        cudaFuncSetAttribute(straight_tile_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * ST_NBUF * (ST_TILE_WORDS + 256) * 4);
        attr_set = true;
    }
    ProfScope prof(p, m);
    const uint32_t *lenq = p->d_lenq + (size_t)m * nt;
    const int nx = p->n_xslices, ny = nt - nx;
    const dim3 gx(bands / warps, nx), gy(bands / warps, ny);
    const int fwd = (m == M_SF);
    if (soft) {
        straight_tile_kernel<true><<<gx, warps * 32, smem, p->stream>>>(p->V, p->S_line, p->d_B, p->d_IJ, p->d_tlist, lenq, p->w.ct[m], p->log2_n, fwd);
        straight_rows_kernel<true><<<gy, warps * 32, 0, p->stream>>>(p->V, p->S_line, p->d_B, p->d_IJ, p->d_tlist + nx, lenq, p->w.ct[m], p->log2_n, fwd);
    } else {
        straight_tile_kernel<false><<<gx, warps * 32, smem, p->stream>>>(p->V, nullptr, p->d_B, p->d_IJ, p->d_tlist, lenq, p->w.ct[m], p->log2_n, fwd);
        straight_rows_kernel<false><<<gy, warps * 32, 0, p->stream>>>(p->V, nullptr, p->d_B, p->d_IJ, p->d_tlist + nx, lenq, p->w.ct[m], p->log2_n, fwd);
    }
    return 2;
}
