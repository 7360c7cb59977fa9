// Obstacle rendering: vehicle footprint x obstacle image -> bit-packed
// collision volume C and uint8 soft volume S.   PAPER.md:88 ("rendering" obstacles into configuration
// space), l.226 (wall at i = 0 / j = 0, toroidal addressing), l.259 (Psi offset), l.338 (section VI),
// l.871 (appendix C: 32 cells per word).  Rasterisation rule: DESIGN R15.
#include "nhp_internal.cuh"

// ---------------------------------------------------------------------------------------------
// E_Theta: which image-pixel offsets (da, db) does the footprint of a pose cover?  Depends only on
// (a - i, b - j, Theta).  One thread per (Theta, db, da); 32 da's are packed with a ballot.
// ---------------------------------------------------------------------------------------------
__global__ void footprint_raster_kernel(uint32_t *__restrict__ E, const uint8_t *__restrict__ mask, int mw, int mh,
                                        long long ouq, long long ovq, const int32_t *__restrict__ rot,
                                        int rad, int side, int sidew)
{
    const int t = blockIdx.z, row = blockIdx.y;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;       // = da + rad
    const int da = col - rad, db = row - rad;
    const int cq = rot[4 * t + 0], sq = rot[4 * t + 1];
    // half-cell units: 2 * (a - i) - 2 Psi0(Theta), eq (16)
    const long long dx2 = 2ll * da - rot[4 * t + 2], dy2 = 2ll * db - rot[4 * t + 3];
    // world -> vehicle frame: inverse of PAPER.md:86, Q14 cos / sin, result in 2^-15 cells
    const long long uq = dx2 * cq + dy2 * sq, vq = -dx2 * sq + dy2 * cq;
    const long long pp = (uq + ouq + 16384) >> 15, qq = (vq + ovq + 16384) >> 15;   // floor
    bool cov = col < side && pp >= 0 && pp < mw && qq >= 0 && qq < mh && mask[qq * mw + pp] != 0;
    const unsigned bits = __ballot_sync(0xffffffffu, cov);
    if ((threadIdx.x & 31) == 0 && (col >> 5) < sidew) E[((size_t)t * side + row) * sidew + (col >> 5)] = bits;
}

int launch_footprint_raster(nhp_planner *p, int mw, int mh, int64_t ouq, int64_t ovq)
{
    dim3 grid(p->sidew, p->side, p->nt), block(32);
    ProfScope prof(p, 10);
    footprint_raster_kernel<<<grid, block, 0, p->stream>>>(p->d_E, p->d_mask, mw, mh, ouq, ovq, p->d_rot, p->rad,
                                                          p->side, p->sidew);
    return 1;
}

// ---------------------------------------------------------------------------------------------
// H = hard | wall as bit rows.  PAPER.md:226: "we insert a single cell hard obstacle wall in each
// spatial dimension (at i = 0 and j = 0)".
// ---------------------------------------------------------------------------------------------
__global__ void pack_hard_kernel(uint32_t *__restrict__ H, const uint8_t *__restrict__ hard, int n)
{
    const int b = blockIdx.y, a = blockIdx.x * blockDim.x + threadIdx.x;
    const bool h = hard[(size_t)b * n + a] != 0 || a == 0 || b == 0;
    const unsigned bits = __ballot_sync(0xffffffffu, h);
    if ((threadIdx.x & 31) == 0) H[(size_t)b * (n >> 5) + (a >> 5)] = bits;
}

// ---------------------------------------------------------------------------------------------
// Run decomposition of E_Theta (host, once per footprint): every row db of E_Theta is a union of runs
// [da_lo, da_lo + len) of covered offsets (one run per row for a convex footprint, several for an
// arbitrary mask).  OR / max over a run of any length is two look-ups in a sparse table of the image
// rows: with k = floor(log2 len), T_k[a] = op(image[a .. a + 2^k - 1]) and
//     op(image[x .. x + len - 1]) = op(T_k[x], T_k[x + len - 2^k])
// (toroidal in a).  A pose then costs 2 look-ups per footprint ROW instead of one per footprint PIXEL.
// ---------------------------------------------------------------------------------------------
int finish_footprint(nhp_planner *p)
{
    const int nt = p->nt, side = p->side, sidew = p->sidew, rad = p->rad;
    std::vector<uint32_t> E((size_t)nt * side * sidew);
    if (cudaMemcpyAsync(E.data(), p->d_E, sizeof(uint32_t) * E.size(), cudaMemcpyDeviceToHost, p->stream) != cudaSuccess) return NHP_E_CUDA;
    if (cudaStreamSynchronize(p->stream) != cudaSuccess) return NHP_E_CUDA;
    std::vector<int4> runs;
    std::vector<int32_t> off(nt + 1, 0);
    int maxk = 0, maxruns = 0;
    for (int t = 0; t < nt; t++) {
        off[t] = (int32_t)runs.size();
        for (int r = 0; r < side; r++) {
            const uint32_t *row = &E[((size_t)t * side + r) * sidew];
            int c = 0;
            while (c < side) {
                if (!((row[c >> 5] >> (c & 31)) & 1u)) { c++; continue; }
                int e = c;
                while (e < side && ((row[e >> 5] >> (e & 31)) & 1u)) e++;
                const int len = e - c;
                int k = 0;
                while ((2 << k) <= len) k++;
                runs.push_back(make_int4(r - rad, c - rad, len - (1 << k), k));      // db, da_lo, second look-up offset, level
                maxk = k > maxk ? k : maxk;
                c = e;
            }
        }
        const int cnt = (int)runs.size() - off[t];
        maxruns = cnt > maxruns ? cnt : maxruns;
    }
    off[nt] = (int32_t)runs.size();
    if (runs.empty()) runs.push_back(make_int4(0, 0, 0, 0));
    // the tables live in the caller's workspace, sized at creation for nhp_limits.max_footprint_radius
    if (runs.size() > p->cap_runs || maxk + 1 > p->cap_levels) return NHP_E_BUFFER;
    p->n_levels = maxk + 1;
    p->max_runs = maxruns;
    if (cudaMemcpyAsync(p->d_runs, runs.data(), sizeof(int4) * runs.size(), cudaMemcpyHostToDevice, p->stream) != cudaSuccess) return NHP_E_CUDA;
    if (cudaMemcpyAsync(p->d_run_off, off.data(), sizeof(int32_t) * (nt + 1), cudaMemcpyHostToDevice, p->stream) != cudaSuccess) return NHP_E_CUDA;
    if (cudaStreamSynchronize(p->stream) != cudaSuccess) return NHP_E_CUDA;
    return NHP_OK;
}

// ---------------------------------------------------------------------------------------------
// Sparse tables of the image rows.  One block per image row b.
//   hard: Hk[k][b][w], bit a of level k = OR of H[b][a .. a + 2^k - 1]      (level 0 = H, written by pack_hard_kernel)
//   soft: Mk[k][b][a]        = max of soft[b][a .. a + 2^k - 1]
// ---------------------------------------------------------------------------------------------
__global__ void hard_levels_kernel(uint32_t *__restrict__ Hk, int n, int levels)
{
    extern __shared__ uint32_t sm[];                 // [2][nw]
    const int nw = n >> 5, mw = nw - 1, b = blockIdx.x;
    const size_t lvl = (size_t)n * nw;
    uint32_t *cur = sm, *nxt = sm + nw;
    for (int w = threadIdx.x; w < nw; w += blockDim.x) cur[w] = Hk[(size_t)b * nw + w];
    __syncthreads();
    for (int k = 1; k < levels; k++) {
        const int s = 1 << (k - 1);
        for (int w = threadIdx.x; w < nw; w += blockDim.x) {
            uint32_t sh;
            if (s < 32) sh = __funnelshift_r(cur[w], cur[(w + 1) & mw], s);
            else sh = cur[(w + (s >> 5)) & mw];
            const uint32_t v = cur[w] | sh;
            nxt[w] = v;
            Hk[k * lvl + (size_t)b * nw + w] = v;
        }
        __syncthreads();
        uint32_t *t = cur; cur = nxt; nxt = t;
    }
}

__global__ void soft_levels_kernel(uint32_t *__restrict__ Mk, const uint8_t *__restrict__ soft, int n, int levels)
{
    extern __shared__ uint32_t sm[];                 // [2][n/4]
    const int nq = n >> 2, mq = nq - 1, b = blockIdx.x;
    const size_t lvl = (size_t)n * nq;
    uint32_t *cur = sm, *nxt = sm + nq;
    const uint32_t *src = (const uint32_t *)(soft + (size_t)b * n);
    for (int q = threadIdx.x; q < nq; q += blockDim.x) { cur[q] = src[q]; Mk[(size_t)b * nq + q] = src[q]; }
    __syncthreads();
    for (int k = 1; k < levels; k++) {
        const int s = 1 << (k - 1);
        for (int q = threadIdx.x; q < nq; q += blockDim.x) {
            uint32_t sh;
            if (s < 4) sh = __funnelshift_r(cur[q], cur[(q + 1) & mq], 8 * s);
            else sh = cur[(q + (s >> 2)) & mq];
            const uint32_t v = __vmaxu4(cur[q], sh);
            nxt[q] = v;
            Mk[k * lvl + (size_t)b * nq + q] = v;
        }
        __syncthreads();
        uint32_t *t = cur; cur = nxt; nxt = t;
    }
}

// ---------------------------------------------------------------------------------------------
// Collision volume: C[Theta][j][i] = OR over the runs of E_Theta of H[(j+db)&M][(i+da_lo .. )&M], 32 poses per
// thread-word.  Block = 8 rows j x 32 words of one Theta slice (or the whole row if narrower).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t window32(const uint32_t *__restrict__ row, int x, int mw)
{
    const int w0 = (x >> 5) & mw;
    return __funnelshift_r(__ldg(row + w0), __ldg(row + ((w0 + 1) & mw)), x & 31);
}

__global__ void __launch_bounds__(256) render_collision_kernel(uint32_t *__restrict__ C, const uint32_t *__restrict__ Hk,
                                                              const int4 *__restrict__ runs, const int32_t *__restrict__ run_off, int n)
{
    extern __shared__ int4 srun[];
    const int nw = n >> 5, mx = n - 1, mw = nw - 1;
    const int t = blockIdx.z;
    const int r0 = run_off[t], cnt = run_off[t + 1] - r0;
    for (int k = threadIdx.x + threadIdx.y * blockDim.x; k < cnt; k += blockDim.x * blockDim.y) srun[k] = runs[r0 + k];
    __syncthreads();
    const int iw = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    if (iw >= nw) return;
    const size_t lvl = (size_t)n * nw;
    uint32_t acc = 0;
    for (int k = 0; k < cnt; k++) {
        const int4 r = srun[k];                                  // db, da_lo, second offset, level
        const uint32_t *row = Hk + r.w * lvl + (size_t)((j + r.x) & mx) * nw;
        const int x = (iw << 5) + r.y;
        acc |= window32(row, x, mw) | window32(row, x + r.z, mw);
    }
    if (j == 0) acc = 0xffffffffu;                               // wall
    if (iw == 0) acc |= 1u;
    C[((size_t)t * n + j) * nw + iw] = acc;
}

// ---------------------------------------------------------------------------------------------
// Soft volume: S = clamp(max over E_Theta of soft, 16, 255) (DESIGN R16), sixteen poses per thread.
// ---------------------------------------------------------------------------------------------
// 16 consecutive bytes of an image row starting at byte `a` (toroidal), as four words: two aligned 16-byte loads cover
// the window, WS = (a & 15) >> 2 (the same for every thread of a run, so the caller branches on it uniformly)
template <int WS>
__device__ __forceinline__ uint4 window16(const uint4 *__restrict__ row, int a, int mQ)
{
    const int Q0 = (a >> 4) & mQ;
    const uint4 lo = __ldg(row + Q0), hi = __ldg(row + ((Q0 + 1) & mQ));
    const uint32_t w[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
    const int bs = (a & 3) * 8;
    return make_uint4(__funnelshift_r(w[WS], w[WS + 1], bs), __funnelshift_r(w[WS + 1], w[WS + 2], bs),
                      __funnelshift_r(w[WS + 2], w[WS + 3], bs), __funnelshift_r(w[WS + 3], w[WS + 4], bs));
}

// Byte-wise maximum without the (emulated, ~9 instructions) __vmaxu4: the running maximum is kept as two words of
// 16-bit lanes (even bytes, odd bytes); the two windows of a run cost four PRMT and two packed three-input 16-bit max
// ops (VIMNMX3.S16x2; the lanes are <= 255, so the signed form is exact) per word.
struct Max16 { uint32_t e[4], o[4]; };

__device__ __forceinline__ void max16_add(Max16 &m, int k, uint32_t x, uint32_t y)
{
    m.e[k] = __vimax3_s16x2(m.e[k], __byte_perm(x, 0u, 0x4240), __byte_perm(y, 0u, 0x4240));     // bytes 0, 2 -> 16-bit lanes
    m.o[k] = __vimax3_s16x2(m.o[k], __byte_perm(x, 0u, 0x4341), __byte_perm(y, 0u, 0x4341));     // bytes 1, 3
}

__device__ __forceinline__ uint4 soft_window(const uint4 *__restrict__ row, int a, int mQ)
{
    switch ((a & 15) >> 2) {                                     // uniform over the block: a = 16 iQ + (run constant)
    case 0: return window16<0>(row, a, mQ);
    case 1: return window16<1>(row, a, mQ);
    case 2: return window16<2>(row, a, mQ);
    default: return window16<3>(row, a, mQ);
    }
}

// Area / orientation penalty ("any additional area and orientation related penalties", Figure 19 l.463;
// reading DESIGN R28) on four rendered soft values packed in a word: dir = preferred heading of the pose's own pixel in 1/256
// turns, pen = Q4.4 factor paid in full when facing the opposite way, h = heading of the plane in 1/256 turns.
//   delta = circular distance of h and dir (0 .. 128),  f = 16 + (((pen - 16) * 2 delta + 128) >> 8),  S <- min(255, (S f + 8) >> 4)
__device__ __forceinline__ uint32_t lane_penalty4(uint32_t s4, uint32_t dir4, uint32_t pen4, int h)
{
    uint32_t out = 0;
#pragma unroll
    for (int b = 0; b < 4; b++) {
        const int s = (s4 >> (8 * b)) & 255, dir = (dir4 >> (8 * b)) & 255, pen = max(16, (int)((pen4 >> (8 * b)) & 255));
        const int d = (h - dir) & 255, delta = min(d, 256 - d);
        const int f = 16 + (((pen - 16) * 2 * delta + 128) >> 8);
        out |= (uint32_t)min(255, (s * f + 8) >> 4) << (8 * b);
    }
    return out;
}

// Sixteen poses per thread: per run two look-ups of 16 bytes each (four aligned 16-byte loads) instead of sixteen 4-byte
// loads, and a quarter of the per-run bookkeeping per pose.  LANE: the penalty of R28 is applied to the sixteen values before
// the one store (lane_dir / lane_pen: the N x N lane map, sixteen pixels per uint4).
template <bool LANE>
__global__ void __launch_bounds__(256) render_soft_kernel(uint4 *__restrict__ S16, const uint4 *__restrict__ Mk,
                                                         const int4 *__restrict__ runs, const int32_t *__restrict__ run_off, int n,
                                                         const uint4 *__restrict__ lane_dir, const uint4 *__restrict__ lane_pen, int log2_nt)
{
    extern __shared__ int4 srun[];
    const int nQ = n >> 4, mx = n - 1, mQ = nQ - 1;
    const int t = blockIdx.z;
    const int r0 = run_off[t], cnt = run_off[t + 1] - r0;
    for (int k = threadIdx.x + threadIdx.y * blockDim.x; k < cnt; k += blockDim.x * blockDim.y) srun[k] = runs[r0 + k];
    __syncthreads();
    const int iQ = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    if (iQ >= nQ) return;
    const size_t lvl = (size_t)n * nQ;
    Max16 acc;
#pragma unroll
    for (int e = 0; e < 4; e++) acc.e[e] = acc.o[e] = 0x00100010u;               // >= 16 = 1.0
    for (int k = 0; k < cnt; k++) {
        const int4 r = srun[k];                                  // db, da_lo, second look-up offset, level
        const uint4 *row = Mk + r.w * lvl + (size_t)((j + r.x) & mx) * nQ;
        const int a = (iQ << 4) + r.y;
        const uint4 x = soft_window(row, a, mQ), y = soft_window(row, a + r.z, mQ);
        max16_add(acc, 0, x.x, y.x); max16_add(acc, 1, x.y, y.y); max16_add(acc, 2, x.z, y.z); max16_add(acc, 3, x.w, y.w);
    }
    uint4 s = make_uint4(acc.e[0] | (acc.o[0] << 8), acc.e[1] | (acc.o[1] << 8), acc.e[2] | (acc.o[2] << 8), acc.e[3] | (acc.o[3] << 8));
    if (LANE) {
        const uint4 d = lane_dir[(size_t)j * nQ + iQ], q = lane_pen[(size_t)j * nQ + iQ];
        const int h = (t << 8) >> log2_nt;                       // floor(256 Theta / N_theta)
        s = make_uint4(lane_penalty4(s.x, d.x, q.x, h), lane_penalty4(s.y, d.y, q.y, h), lane_penalty4(s.z, d.z, q.z, h),
                       lane_penalty4(s.w, d.w, q.w, h));
    }
    S16[((size_t)t * n + j) * nQ + iQ] = s;
}

int launch_render(nhp_planner *p, bool soft)
{
    const int n = p->n, nw = n / 32, nq = n / 4;
    int launches = 0;
    {
        ProfScope prof(p, 10);
        pack_hard_kernel<<<dim3(n / 32, n), 32, 0, p->stream>>>(p->d_Hk, p->d_hard, n);
        hard_levels_kernel<<<n, nw < 32 ? 32 : nw, sizeof(uint32_t) * 2 * nw, p->stream>>>(p->d_Hk, n, p->n_levels);
        launches += 2;
        if (soft) {
            soft_levels_kernel<<<n, nq < 256 ? nq : 256, sizeof(uint32_t) * 2 * nq, p->stream>>>((uint32_t *)p->d_Mk, p->d_soft, n, p->n_levels);
            launches++;
        }
    }
    const size_t smem = sizeof(int4) * (size_t)(p->max_runs > 0 ? p->max_runs : 1);
    {
        ProfScope prof(p, 6);
        const dim3 block(nw < 32 ? nw : 32, 8);
        render_collision_kernel<<<dim3(nw / block.x, n / 8, p->nt), block, smem, p->stream>>>(p->C, p->d_Hk, p->d_runs, p->d_run_off, n);
        launches++;
    }
    if (soft) {
        ProfScope prof(p, 7);
        const int nQ = n / 16;
        const dim3 block(nQ < 32 ? nQ : 32, 8);
        const dim3 grid(nQ / block.x, n / 8, p->nt);
        if (p->have_lane) render_soft_kernel<true><<<grid, block, smem, p->stream>>>((uint4 *)p->S, (const uint4 *)p->d_Mk, p->d_runs, p->d_run_off, n,
                                                                                   (const uint4 *)p->d_lane_dir, (const uint4 *)p->d_lane_pen, p->log2_nt);
        else render_soft_kernel<false><<<grid, block, smem, p->stream>>>((uint4 *)p->S, (const uint4 *)p->d_Mk, p->d_runs, p->d_run_off, n,
                                                                       nullptr, nullptr, p->log2_nt);
        launches++;
        launches += launch_soft_layouts(p);
    }
    return launches;
}
