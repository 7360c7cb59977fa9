// Integer-pipe micro-benchmark (nhp_microbench_alu, include/nhplan.h): the peak behind bench.py's `alu` line,
// DESIGN.md section 6.7.  Every step of every sweep (Insert 5) is made of VIADDMNMX operations
// (nhp_arrive / nhp_keep / nhp_gate); this kernel issues nothing else, in `CH` independent dependency chains per
// thread, 8 warps per SM sub-partition, and is timed with CUDA events on the handle's stream.
#include "nhp_internal.cuh"

namespace {

constexpr int MB_ITERS = 4096, MB_THREADS = 256, MB_CTAS_PER_SM = 4;

template <int CH>
__global__ void __launch_bounds__(MB_THREADS) alu_chain_kernel(uint32_t *__restrict__ sink, uint32_t w, uint32_t u)
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
    if (x == 0xdeadbeefu) sink[0] = x;                // keeps the chains alive; never true for the arguments passed
}

template <int CH>
void launch(int ctas, uint32_t *sink, cudaStream_t s)
{
    alu_chain_kernel<CH><<<ctas, MB_THREADS, 0, s>>>(sink, 3u, 0x7fff0000u);
}

}  // namespace

extern "C" int nhp_microbench_alu(nhp_planner *p, int chains, double *lane_ops_per_s, int *sms)
{
    if (!p || chains < 1 || chains > 8 || !lane_ops_per_s) return NHP_E_ARG;
    DeviceGuard guard(p);
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, p->device) != cudaSuccess) return NHP_E_CUDA;
    const int ctas = n_sm * MB_CTAS_PER_SM;
    uint32_t *sink = (uint32_t *)p->d_status + NHP_STATUS_WORDS - 1;       // never written (see the kernel)
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return NHP_E_CUDA;
    float best = 1e30f;
    for (int rep = 0; rep < 4; rep++) {                                  // first repetition warms up
        cudaEventRecord(e0, p->stream);
        switch (chains) {
            case 1: launch<1>(ctas, sink, p->stream); break;
            case 2: launch<2>(ctas, sink, p->stream); break;
            case 3: launch<3>(ctas, sink, p->stream); break;
            case 4: launch<4>(ctas, sink, p->stream); break;
            case 5: launch<5>(ctas, sink, p->stream); break;
            case 6: launch<6>(ctas, sink, p->stream); break;
            case 7: launch<7>(ctas, sink, p->stream); break;
            default: launch<8>(ctas, sink, p->stream); break;
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
