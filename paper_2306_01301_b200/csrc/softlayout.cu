// Curve-major copies of the soft volume S (second half).
//
// A sweep kernel walks along curves; its value volume V is staged tile by tile (sweep.cu, straight.cu), but the
// soft multiplier S is one BYTE per vertex, too narrow to stage the same way (cp.async moves >= 4 bytes, and a warp
// reading one byte per plane fetches a 32-byte sector for it).  So the renderer also writes S in the order the
// sweeps consume it:
//   S_left [y'][x' / 32][Theta / 4][x' % 32][Theta % 4] = S[Theta][(y' + beta3(Theta)) & M][(x' + beta0(Theta)) & M]     left-turn curves, eq (18)
//   S_right[y'][x' / 32][Theta / 4][x' % 32][Theta % 4] = S[Theta][(y' + beta1(Theta)) & M][(x' + beta2(Theta)) & M]     right-turn curves, eq (18)
//       (tile-major: the four bytes of four consecutive planes of one curve are one word, the 32 curves of a turn tile lie next to
//       each other, so a warp of the tile kernel reads one 128-byte line per four planes)
//   S_line [Theta][x' / 32][y' / 32][(y' / 16) % 2][x' % 32][y' % 16] = S at the vertex eq (23) gives for (x', y', Theta)     straight lines
//       (the 16 bytes a thread reads at once next to those of the 31 other lines of its warp)
// Same bytes, same traffic per pose-update (1 B), three more volumes of N_R bytes in the caller's workspace.
#include "nhp_internal.cuh"

// One block = 32 neighbouring curves (x' = x0 .. x0 + 31 at one y') of one turn family, lane = curve.  A warp produces the words
// j = warp, warp + nwarps, ...: four byte loads (the curve's vertices in the planes 4 j .. 4 j + 3, each a 32-byte row segment for
// the warp) packed into one word, stored as one 128-byte line -- no shared memory, no barrier.
__global__ void __launch_bounds__(256) soft_turn_layout_kernel(uint8_t *__restrict__ Sout, const uint8_t *__restrict__ S,
                                                              const int16_t *__restrict__ beta, int log2_n, int nt, int qa, int qb)
{
    const int mx = (1 << log2_n) - 1, mt = nt - 1, quarter = nt >> 2;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int x0 = blockIdx.x << 5, yp = blockIdx.y;
    uint32_t *out = (uint32_t *)Sout + (((size_t)yp << (log2_n - 5)) + blockIdx.x) * ((size_t)nt * 8);
    for (int j = warp; j < (nt >> 2); j += nwarps) {
        uint32_t word = 0;
#pragma unroll
        for (int e = 0; e < 4; e++) {
            const int t = 4 * j + e;
            const int ba = beta[(t + qa * quarter) & mt], bb = beta[(t + qb * quarter) & mt];
            word |= (uint32_t)S[((((size_t)t << log2_n) + ((yp + bb) & mx)) << log2_n) + ((x0 + ba + lane) & mx)] << (8 * e);
        }
        out[j * 32 + lane] = word;
    }
}

// The same for grids of at least 128 cells per side, four tiles (128 neighbouring curves) per block and four curves per lane: per
// plane two aligned 4-byte loads (wrapped on the torus per lane) and a funnel shift give the lane's four bytes whatever the
// alignment of the row segment; the 4 x 4 bytes of four planes are transposed in registers (eight PRMT) into the four output
// words, stored as one 16-byte piece.  Four times fewer load instructions per byte than soft_turn_layout_kernel.
__global__ void __launch_bounds__(256) soft_turn_layout4_kernel(uint8_t *__restrict__ Sout, const uint8_t *__restrict__ S,
                                                               const int16_t *__restrict__ beta, int log2_n, int nt, int qa, int qb)
{
    const int mx = (1 << log2_n) - 1, mt = nt - 1, quarter = nt >> 2;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int x0 = blockIdx.x << 7, yp = blockIdx.y;
    // tile (yp, 4 blockIdx.x + lane / 8), word j, curves 4 (lane % 8) .. + 3
    uint32_t *out = (uint32_t *)Sout + (((size_t)yp << (log2_n - 5)) + 4 * blockIdx.x + (lane >> 3)) * ((size_t)nt * 8) + 4 * (lane & 7);
    for (int j = warp; j < (nt >> 2); j += nwarps) {
        uint32_t W[4];
#pragma unroll
        for (int e = 0; e < 4; e++) {
            const int t = 4 * j + e;
            const int ba = beta[(t + qa * quarter) & mt], bb = beta[(t + qb * quarter) & mt];
            const uint8_t *row = S + ((((size_t)t << log2_n) + ((yp + bb) & mx)) << log2_n);
            const int c = (x0 + ba + 4 * lane) & mx, c0 = c & ~3;           // (c & 3 is the same in every lane: N is a multiple of 4)
            const uint32_t w0 = *(const uint32_t *)(row + c0), w1 = *(const uint32_t *)(row + ((c0 + 4) & mx));
            W[e] = __funnelshift_r(w0, w1, 8 * (c & 3));
        }
        const uint32_t t0 = __byte_perm(W[0], W[1], 0x5140), t1 = __byte_perm(W[2], W[3], 0x5140);
        const uint32_t t2 = __byte_perm(W[0], W[1], 0x7362), t3 = __byte_perm(W[2], W[3], 0x7362);
        *(uint4 *)(out + j * 32) = make_uint4(__byte_perm(t0, t1, 0x5410), __byte_perm(t0, t1, 0x7632), __byte_perm(t2, t3, 0x5410),
                                              __byte_perm(t2, t3, 0x7632));
    }
}

// One block = a 32 x 32 tile (x', y') of one Theta slice: the bytes of 32 neighbouring lines x' = 32 band + l at the steps
// y' = 32 T + 16 h + e go to S_line[Theta][band][T][h][l][e] -- the 16 bytes (e) a thread of the straight kernels reads at once next to
// those of the other 31 lines of its warp, so a warp's two loads per tile are 512 contiguous bytes each.
__global__ void __launch_bounds__(256) soft_line_layout_kernel(uint8_t *__restrict__ Sout, const uint8_t *__restrict__ S,
                                                              const int16_t *__restrict__ B, const uint8_t *__restrict__ IJ, int log2_n)
{
    __shared__ __align__(16) uint8_t tile[32][48];              // [line][step], 16-byte aligned rows
    const int n = 1 << log2_n, mx = n - 1;
    const int t = blockIdx.z, x0 = blockIdx.x << 5, y0 = blockIdx.y << 5;
    const int lane = threadIdx.x, ty = threadIdx.y;
    const int16_t *Bt = B + (size_t)t * n;
    const uint8_t *St = S + ((size_t)t << (2 * log2_n));
    if ((IJ[t] & 1) == 0) {
        // eq (23), I = 0: (i, j) = (y', (x' + B(y')) & M): lane = y' is the memory-fast axis
        const int y = y0 + lane, b = Bt[y];
        for (int r = ty; r < 32; r += 8) tile[r][lane] = St[((size_t)((x0 + r + b) & mx) << log2_n) + y];
    } else {
        // I = 1: (i, j) = ((x' + B(y')) & M, y'): lane = x' is the memory-fast axis
        for (int r = ty; r < 32; r += 8) {
            const int y = y0 + r;
            tile[lane][r] = St[((size_t)y << log2_n) + ((x0 + lane + Bt[y]) & mx)];
        }
    }
    __syncthreads();
    const int k = ty * 32 + lane;                               // 64 threads write one 16-byte piece each: k = 32 h + l
    if (k < 64) {
        const int h = k >> 5, l = k & 31;
        uint4 *out = (uint4 *)(Sout + ((size_t)t << (2 * log2_n)) + (((size_t)blockIdx.x << (log2_n - 5)) + blockIdx.y) * 1024);
        out[k] = *(const uint4 *)&tile[l][16 * h];
    }
}

int launch_soft_layouts(nhp_planner *p)
{
    const int n = p->n, nt = p->nt;
    if (n >= 128) {
        soft_turn_layout4_kernel<<<dim3(n / 128, n), 256, 0, p->stream>>>(p->S_left, p->S, p->d_beta, p->log2_n, nt, 0, 3);
        soft_turn_layout4_kernel<<<dim3(n / 128, n), 256, 0, p->stream>>>(p->S_right, p->S, p->d_beta, p->log2_n, nt, 2, 1);
    } else {
        soft_turn_layout_kernel<<<dim3(n / 32, n), 256, 0, p->stream>>>(p->S_left, p->S, p->d_beta, p->log2_n, nt, 0, 3);
        soft_turn_layout_kernel<<<dim3(n / 32, n), 256, 0, p->stream>>>(p->S_right, p->S, p->d_beta, p->log2_n, nt, 2, 1);
    }
    soft_line_layout_kernel<<<dim3(n / 32, n / 32, nt), dim3(32, 8), 0, p->stream>>>(p->S_line, p->S, p->d_B, p->d_IJ, p->log2_n);
    return 3;
}

// function attributes are per device: set for the handle's device at creation (nhp_planner_create)
int set_softlayout_attributes()
{
    return NHP_OK;                 // (no kernel of this file needs more than the default shared memory any more)
}
