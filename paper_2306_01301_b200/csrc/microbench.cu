// Integer-pipe micro-benchmark (nhp_microbench_alu, include/nhplan.h): the peak behind bench.py's `alu` line,
// DESIGN.md section 6.7.  Every step of every sweep (Insert 5) is made of VIADDMNMX operations
// (nhp_arrive / nhp_keep / nhp_gate); this kernel issues nothing else, in `CH` independent dependency chains per
// thread, 8 warps per SM sub-partition, and is timed with CUDA events on the handle's stream.
#include "nhp_internal.cuh"
#include "../../include/nhplan_probe.h"

// The probes' own sink word (device code names it directly): written only if an impossible value turns up, which keeps the
// measured instructions alive without touching anything of the planner's.
#pragma nv_diag_suppress 550                      /* "set but never used": that is the point of a sink */
static __device__ uint32_t probe_sink;

namespace {

constexpr int MB_ITERS = 4096, MB_THREADS = 256, MB_CTAS_PER_SM = 4;

template <int CH>
__global__ void __launch_bounds__(MB_THREADS) alu_chain_kernel(uint32_t w, uint32_t u)
{
    uint32_t t[CH];
#pragma unroll
    for (int c = 0; c < CH; c++) t[c] = threadIdx.x + c;
#pragma unroll 1
    for (int it = 0; it < MB_ITERS; it += 8) {
#pragma unroll
        for (int k = 0; k < 8; k++) {
#pragma unroll
            for (int c = 0; c < CH; c++) t[c] = nhp_arrive(t[c], w, u + k);      // min(t + w, u'): one VIADDMNMX
        }
    }
    uint32_t x = 0;
#pragma unroll
    for (int c = 0; c < CH; c++) x ^= t[c];
    if (x == 0xdeadbeefu) probe_sink = x;               // keeps the chains alive; never true for the arguments passed
}

template <int CH>
void launch(int ctas, cudaStream_t s)
{
    alu_chain_kernel<CH><<<ctas, MB_THREADS, 0, s>>>(3u, 0x7fff0000u);
}

}  // namespace

extern "C" int nhp_microbench_alu(nhp_planner *p, int chains, double *lane_ops_per_s, int *sms)
{
    if (!p || chains < 1 || chains > 8 || !lane_ops_per_s) return NHP_E_ARG;
    DeviceGuard guard(p);
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, p->device) != cudaSuccess) return NHP_E_CUDA;
    const int ctas = n_sm * MB_CTAS_PER_SM;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return NHP_E_CUDA;
    float best = 1e30f;
    for (int rep = 0; rep < 4; rep++) {                                  // first repetition warms up
        cudaEventRecord(e0, p->stream);
        switch (chains) {
            case 1: launch<1>(ctas, p->stream); break;
            case 2: launch<2>(ctas, p->stream); break;
            case 3: launch<3>(ctas, p->stream); break;
            case 4: launch<4>(ctas, p->stream); break;
            case 5: launch<5>(ctas, p->stream); break;
            case 6: launch<6>(ctas, p->stream); break;
            case 7: launch<7>(ctas, p->stream); break;
            default: launch<8>(ctas, p->stream); break;
        }
        cudaEventRecord(e1, p->stream);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return NHP_E_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    p->launches += 4;
    const double ops = (double)ctas * MB_THREADS * (double)MB_ITERS * chains;
    *lane_ops_per_s = ops / ((double)best * 1e-3);
    if (sms) *sms = n_sm;
    return NHP_OK;
}

// ---------------------------------------------------------------------------------------------
// Read probes behind the roofline discussion of DESIGN.md section 6: nothing but the loads of the value volume, in the
// access patterns of the three sweep kernels, 32 loads per thread in flight at a time.
//   pattern 0  linear: every warp reads 4 KB contiguous chunks
//   pattern 1  rows-like (straight_rows_kernel): a warp walks a band of one slice, tile = 32 rows x 128 bytes at a 4 N-byte stride
//   pattern 2  x-rows-like (straight_xl_kernel): a warp walks along the rows, tile = 32 rows x 128 bytes, next tile 128 bytes on
//   pattern 3  turn-like (turn_tile_kernel): CTA = N_theta / 32 warps, warp s reads planes 32 s .. 32 s + 31 of one tile
// ---------------------------------------------------------------------------------------------
template <int MODE>
__global__ void read_probe_kernel(const uint32_t *__restrict__ V, int log2_n, int nt)
{
    const int lane = threadIdx.x & 31, n = 1 << log2_n, NT = n >> 5;
    const size_t gw = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    uint32_t acc = 0;
    const int tiles = MODE == 3 ? 1 : NT;
    for (int T = 0; T < tiles; T++) {
        uint32_t u[32];
        const uint32_t *p;
        size_t stride;
        if (MODE == 0) { p = V + (gw * NT + T) * 1024 + lane; stride = 32; }
        else if (MODE == 1) { const size_t b = gw % NT, t = gw / NT; p = V + (t << (2 * log2_n)) + ((size_t)(32 * T) << log2_n) + 32 * b + lane; stride = (size_t)n; }
        else if (MODE == 2) { const size_t b = gw % NT, t = gw / NT; p = V + (t << (2 * log2_n)) + ((size_t)(32 * b) << log2_n) + 32 * T + lane; stride = (size_t)n; }
        else { const size_t s = threadIdx.x >> 5, bx = blockIdx.x % NT, yp = blockIdx.x / NT; p = V + ((32 * s) << (2 * log2_n)) + (yp << log2_n) + 32 * bx + lane; stride = (size_t)1 << (2 * log2_n); }
#pragma unroll
        for (int k = 0; k < 32; k++) u[k] = p[k * stride];
#pragma unroll
        for (int k = 0; k < 32; k++) acc ^= u[k];
    }
    if (acc == 0x12345678u) probe_sink = acc;             // keeps the loads alive; a volume of costs never XORs to this in every thread
}

extern "C" int nhp_microbench_read(nhp_planner *p, int pattern, double *bytes_per_s)
{
    if (!p || pattern < 0 || pattern > 3 || !bytes_per_s) return NHP_E_ARG;
    DeviceGuard guard(p);
    const int n = p->n, nt = p->nt, NT = n / 32;
    const size_t nr = (size_t)n * n * nt, warps = nr / 1024 / (pattern == 3 ? 1 : NT);
    const int threads = pattern == 3 ? nt : 128;
    const unsigned blocks = (unsigned)(warps * 32 / threads);
    if (pattern == 3 && nt > 1024) return NHP_E_ARG;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return NHP_E_CUDA;
    float best = 1e30f;
    for (int rep = 0; rep < 4; rep++) {
        cudaEventRecord(e0, p->stream);
        switch (pattern) {
            case 0: read_probe_kernel<0><<<blocks, threads, 0, p->stream>>>(p->V, p->log2_n, nt); break;
            case 1: read_probe_kernel<1><<<blocks, threads, 0, p->stream>>>(p->V, p->log2_n, nt); break;
            case 2: read_probe_kernel<2><<<blocks, threads, 0, p->stream>>>(p->V, p->log2_n, nt); break;
            default: read_probe_kernel<3><<<blocks, threads, 0, p->stream>>>(p->V, p->log2_n, nt); break;
        }
        cudaEventRecord(e1, p->stream);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return NHP_E_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    p->launches += 4;
    *bytes_per_s = 4.0 * (double)nr / ((double)best * 1e-3);
    return NHP_OK;
}
