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

// ---- nhp_soft_from_hard_noalloc: the same two kernels for callers that must not allocate (see include/nhplan.h) -------------------
// Every other call of the library needs a handle, and nhp_planner_create cudaMallocs its tables and the distance transform's
// intermediate image.  This one needs no handle.  Its intermediate image g(y, x') -- the only memory the two kernels touch besides
// their input and outputs -- is the file-scope array below, part of the loaded module on every device that loads the library.
#include <mutex>
#include <stdio.h>

static __device__ __align__(256) int32_t noalloc_g[NHP_NOALLOC_MAX_N * NHP_NOALLOC_MAX_N];      // 4 MiB per device, until the process exits

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex noalloc_mutex;                                     // guards noalloc_g_dev
int32_t *noalloc_g_dev[NOALLOC_MAX_DEVICES];                  // [d] = address of noalloc_g in the memory of device d; nullptr = not asked yet
thread_local char noalloc_error[200] = "";                    // text of the calling thread's last failure

int noalloc_fail(int code, const char *what, cudaError_t e = cudaSuccess)
{
    if (e != cudaSuccess) snprintf(noalloc_error, sizeof(noalloc_error), "%s: %s", what, cudaGetErrorString(e));
    else snprintf(noalloc_error, sizeof(noalloc_error), "%s", what);
    cudaGetLastError();                                       // leave no sticky-looking error behind for the caller's own checks
    return code;
}

// In host code the name `noalloc_g` stands for a host-side shadow of the array, not for anything a kernel can dereference: the
// address a kernel needs is asked from the runtime, once per device, WITH THAT DEVICE CURRENT (each device holds its own copy of
// the array, at its own address).  Allocates nothing.
int noalloc_scratch(int device, int32_t **out)
{
    std::lock_guard<std::mutex> lock(noalloc_mutex);
    if (!noalloc_g_dev[device]) {
        void *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, noalloc_g);
        if (e != cudaSuccess || !ptr) return noalloc_fail(NHP_E_CUDA, "cudaGetSymbolAddress(scratch of nhp_soft_from_hard_noalloc)", e);
        noalloc_g_dev[device] = (int32_t *)ptr;
    }
    *out = noalloc_g_dev[device];
    return NHP_OK;
}

// device that owns a caller's buffer; -1 if it is not plain device memory
int noalloc_device_of(const void *ptr)
{
    cudaPointerAttributes attr{};
    if (cudaPointerGetAttributes(&attr, ptr) != cudaSuccess || attr.type != cudaMemoryTypeDevice) { cudaGetLastError(); return -1; }
    return attr.device;
}
}  // namespace

extern "C" const char *nhp_noalloc_last_error(void) { return noalloc_error; }

extern "C" int nhp_soft_from_hard_noalloc(const uint8_t *hard_dev, int n, double k, uint8_t *soft_dev_out, float *dist_dev_out,
                                          void *cuda_stream)
{
    noalloc_error[0] = 0;
    if (!hard_dev || !soft_dev_out) return noalloc_fail(NHP_E_ARG, "hard_dev / soft_dev_out is NULL");
    if (n < 1) return noalloc_fail(NHP_E_ARG, "n < 1");
    if (n > NHP_NOALLOC_MAX_N) {
        snprintf(noalloc_error, sizeof(noalloc_error), "n = %d is beyond NHP_NOALLOC_MAX_N = %d: the built-in scratch array holds %d x %d "
                 "column distances and cannot grow; use nhp_render_obstacles_dt (caller-sized buffers) for larger images",
                 n, NHP_NOALLOC_MAX_N, NHP_NOALLOC_MAX_N, NHP_NOALLOC_MAX_N);
        return NHP_E_BUFFER;
    }
    if (!(k >= 0.0) || k > 64.0) return noalloc_fail(NHP_E_ARG, "k outside [0, 64]");
    const int device = noalloc_device_of(hard_dev);
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return noalloc_fail(NHP_E_BUFFER, "hard_dev is not device memory");
    if (noalloc_device_of(soft_dev_out) != device || (dist_dev_out && noalloc_device_of(dist_dev_out) != device))
        return noalloc_fail(NHP_E_BUFFER, "soft_dev_out / dist_dev_out is not device memory of the device that owns hard_dev");

    int prev = -1;                                            // the buffers' device is current for the rest of the call
    cudaError_t e = cudaGetDevice(&prev);
    if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
    if (e != cudaSuccess) return noalloc_fail(NHP_E_CUDA, "cudaSetDevice", e);

    int32_t *g = nullptr;
    int rc = noalloc_scratch(device, &g);
    if (rc == NHP_OK) {
        // Nothing in g has to be cleared: the first scan of dt_columns_kernel writes every one of the n x n words (rows of n
        // words, whatever the last call's n was) before anything reads them; words beyond n x n are not touched.
        cudaStream_t stream = (cudaStream_t)cuda_stream;
        dt_columns_kernel<<<(n + 127) / 128, 128, 0, stream>>>(g, hard_dev, n);
        dt_rows_soft_kernel<<<n, n < 256 ? n : 256, sizeof(int32_t) * n, stream>>>(soft_dev_out, dist_dev_out, nullptr, g, n, (float)k);
        e = cudaGetLastError();
        if (e != cudaSuccess) rc = noalloc_fail(NHP_E_CUDA, "kernel launch", e);
    }
    if (prev >= 0 && prev != device) cudaSetDevice(prev);
    return rc;
}
