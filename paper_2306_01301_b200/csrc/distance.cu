// Distance transform of the obstacle image and soft-image synthesis on the device: steps 1-2 of the pipeline
// (section VII l.342: "soft obstacle costs ... some function of the distance"), which the paper runs
// on the CPU before the upload.  Reading DESIGN R17:
//     H    = hard | wall (row 0, column 0), not toroidal
//     d2   = exact squared Euclidean distance to the nearest pixel of H        (integers)
//     d    = sqrt(d2) in float32, round to nearest
//     soft = clamp(rint(16 * (1 + k / (d + 1))), 16, 255), every operation rounded once (no FMA contraction)
// Exact separable form: g(y, x') = distance to the nearest pixel of H in column x', d2(y, x) = min over x' of
// (x - x')^2 + g(y, x')^2.  The image is N x N <= 4096^2 and cache-resident: plain O(N) scans per pixel.
#include "nhp_internal.cuh"

constexpr int DT_FAR = 20000;                    // "no pixel of H in this column" (never happens: row 0 is wall)

// one thread per column: two scans along the column
__global__ void dt_columns_kernel(int32_t *__restrict__ g, const uint8_t *__restrict__ hard, int n)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= n) return;
    int d = DT_FAR;
    for (int y = 0; y < n; y++) {                // nearest pixel of H above or at y
        const bool h = hard[(size_t)y * n + x] != 0 || x == 0 || y == 0;
        d = h ? 0 : min(d + 1, DT_FAR);
        g[(size_t)y * n + x] = d;
    }
    d = DT_FAR;
    for (int y = n - 1; y >= 0; y--) {           // ... or below
        const int up = g[(size_t)y * n + x];
        d = (up == 0) ? 0 : min(d + 1, DT_FAR);
        g[(size_t)y * n + x] = min(up, d);
    }
}

// one block per image row: g(y, .) in shared memory, one thread per pixel (strided), minimum over all columns
__global__ void dt_rows_soft_kernel(uint8_t *__restrict__ soft, float *__restrict__ dist, int32_t *__restrict__ d2_out,
                                    const int32_t *__restrict__ g, int n, float k)
{
    extern __shared__ int32_t sg[];              // g(y, x')^2
    const int y = blockIdx.x;
    for (int a = threadIdx.x; a < n; a += blockDim.x) {
        const int v = g[(size_t)y * n + a];
        sg[a] = v * v;
    }
    __syncthreads();
    for (int x = threadIdx.x; x < n; x += blockDim.x) {
        int best = 0x7fffffff;
        for (int a = 0; a < n; a++) {
            const int dx = x - a;
            best = min(best, dx * dx + sg[a]);
        }
        const float d = __fsqrt_rn((float)best);
        const float v = __fmul_rn(16.0f, __fadd_rn(1.0f, __fdiv_rn(k, __fadd_rn(d, 1.0f))));
        const float r = rintf(v);
        const size_t idx = (size_t)y * n + x;
        soft[idx] = (uint8_t)fminf(fmaxf(r, 16.0f), 255.0f);
        if (dist) dist[idx] = d;
        if (d2_out) d2_out[idx] = best;
    }
}

// d_hard -> d_soft (and the optional outputs); returns the number of kernels launched
int launch_soft_from_hard(nhp_planner *p, float k, float *dist_dev, int32_t *d2_dev)
{
    const int n = p->n;
    ProfScope prof(p, 12);
    dt_columns_kernel<<<(n + 127) / 128, 128, 0, p->stream>>>(p->d_dtg, p->d_hard, n);
    dt_rows_soft_kernel<<<n, n < 256 ? n : 256, sizeof(int32_t) * n, p->stream>>>(p->d_soft, dist_dev, d2_dev, p->d_dtg, n, k);
    return 2;
}
