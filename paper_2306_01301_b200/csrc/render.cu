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
// Collision volume: C[Theta][j][i] = OR over (da, db) in E_Theta of H[(j+db)&M][(i+da)&M], 32 poses
// per thread-word.  A block renders RJ rows of one Theta slice from a shared-memory copy of the
// H rows it needs (RJ + 2 rad rows, wrapped).
// ---------------------------------------------------------------------------------------------
template <int RJ>
__global__ void __launch_bounds__(256) render_collision_kernel(uint32_t *__restrict__ C, const uint32_t *__restrict__ H,
                                                              const uint32_t *__restrict__ E, int n, int rad, int side,
                                                              int sidew)
{
    extern __shared__ uint32_t sm[];
    const int nw = n >> 5, mx = n - 1, mw = nw - 1;
    const int t = blockIdx.y, j0 = blockIdx.x * RJ;
    const int rows = RJ + 2 * rad;
    uint32_t *sE = sm;                       // [side][sidew]
    uint32_t *sH = sm + side * sidew;        // [rows][nw]
    for (int k = threadIdx.x; k < side * sidew; k += blockDim.x) sE[k] = E[(size_t)t * side * sidew + k];
    for (int k = threadIdx.x; k < rows * nw; k += blockDim.x) {
        const int r = k / nw, w = k - r * nw;
        sH[k] = H[(size_t)((j0 - rad + r) & mx) * nw + w];
    }
    __syncthreads();
    for (int k = threadIdx.x; k < RJ * nw; k += blockDim.x) {
        const int jj = k / nw, iw = k - jj * nw;
        uint32_t acc = 0;
        for (int r = 0; r < side; r++) {
            const uint32_t *hrow = sH + (jj + r) * nw;               // image row j + db, db = r - rad
            for (int ew = 0; ew < sidew; ew++) {
                uint32_t bits = sE[r * sidew + ew];
                while (bits) {
                    const int bpos = __ffs(bits) - 1;
                    bits &= bits - 1;
                    const int x = iw * 32 + (ew * 32 + bpos - rad);  // first pixel column a = i + da
                    const int w0 = (x >> 5) & mw;
                    acc |= __funnelshift_r(hrow[w0], hrow[(w0 + 1) & mw], x & 31);
                }
            }
        }
        const int j = j0 + jj;
        if (j == 0) acc = 0xffffffffu;
        if (iw == 0) acc |= 1u;
        C[((size_t)t * n + j) * nw + iw] = acc;
    }
}

// ---------------------------------------------------------------------------------------------
// Soft volume: S = clamp(max over E_Theta of soft, 16, 255) (DESIGN R16), four poses per thread.
// Tile of TX x TY poses with a halo of rad pixels staged in shared memory.
// ---------------------------------------------------------------------------------------------
constexpr int STX = 64, STY = 16;

__global__ void __launch_bounds__(256) render_soft_kernel(uint8_t *__restrict__ S, const uint8_t *__restrict__ soft,
                                                         const uint32_t *__restrict__ E, int n, int rad, int side,
                                                         int sidew)
{
    extern __shared__ uint32_t sm[];
    const int mx = n - 1;
    const int t = blockIdx.z, i0 = blockIdx.x * STX, j0 = blockIdx.y * STY;
    const int pw = ((STX + 2 * rad + 6) >> 2) + 1;            // padded tile width in words
    const int ph = STY + 2 * rad;
    uint32_t *sE = sm;
    uint8_t *sS = (uint8_t *)(sm + side * sidew);            // [ph][pw*4], column 0 <-> image column i0 - rad
    for (int k = threadIdx.x; k < side * sidew; k += blockDim.x) sE[k] = E[(size_t)t * side * sidew + k];
    for (int k = threadIdx.x; k < ph * pw * 4; k += blockDim.x) {
        const int r = k / (pw * 4), c = k - r * (pw * 4);
        sS[k] = soft[(size_t)((j0 - rad + r) & mx) * n + ((i0 - rad + c) & mx)];
    }
    __syncthreads();
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;  // 16 x 16 threads, 4 pixels each
    uint32_t acc = 0x10101010u;                              // >= 16 = 1.0
    const uint32_t *sw = (const uint32_t *)sS;
    for (int r = 0; r < side; r++) {
        const uint32_t *row = sw + (ty + r) * pw;
        for (int ew = 0; ew < sidew; ew++) {
            uint32_t bits = sE[r * sidew + ew];
            while (bits) {
                const int bpos = __ffs(bits) - 1;
                bits &= bits - 1;
                const int c = tx * 4 + ew * 32 + bpos;        // tile column of the first pixel: (i - i0) + da + rad
                const uint32_t lo = row[c >> 2], hi = row[(c >> 2) + 1];
                acc = __vmaxu4(acc, __funnelshift_r(lo, hi, (c & 3) * 8));
            }
        }
    }
    if (i0 + tx * 4 < n)                                     // n = 32: the 64-wide tile wraps onto itself
        *(uint32_t *)(S + ((size_t)t * n + (j0 + ty)) * n + i0 + tx * 4) = acc;
}

int launch_render(nhp_planner *p, bool soft)
{
    const int n = p->n;
    {
        ProfScope prof(p, 10);
        pack_hard_kernel<<<dim3(n / 32, n), 32, 0, p->stream>>>(p->d_H, p->d_hard, n);
    }
    int launches = 1;
    {
        constexpr int RJ = 16;
        ProfScope prof(p, 6);
        const size_t smem = sizeof(uint32_t) * ((size_t)p->side * p->sidew + (size_t)(RJ + 2 * p->rad) * (n / 32));
        cudaFuncSetAttribute(render_collision_kernel<RJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        render_collision_kernel<RJ><<<dim3(n / RJ, p->nt), 256, smem, p->stream>>>(p->C, p->d_H, p->d_E, n, p->rad,
                                                                                   p->side, p->sidew);
        launches++;
    }
    if (soft) {
        const int pw = ((STX + 2 * p->rad + 6) >> 2) + 1, ph = STY + 2 * p->rad;
        const size_t smem = sizeof(uint32_t) * ((size_t)p->side * p->sidew + (size_t)ph * pw);
        cudaFuncSetAttribute(render_soft_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        ProfScope prof(p, 7);
        render_soft_kernel<<<dim3(n < STX ? 1 : n / STX, n / STY, p->nt), 256, smem, p->stream>>>(p->S, p->d_soft, p->d_E, n,
                                                                                   p->rad, p->side, p->sidew);
        launches++;
    }
    return launches;
}
