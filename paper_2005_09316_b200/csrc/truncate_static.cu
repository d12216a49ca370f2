// truncate_static.cu -- woden_truncate_select_static: the Eq 23-24 selection for
// callers that are not allowed to allocate device memory.
//
// Who that is: code running inside someone else's memory budget.  A pipeline stage whose host framework
// owns a fixed device arena, a plug-in called from a region where the allocator is locked, a process
// that shares its GPU under a hard memory quota, or a real-time loop that must not hit the implicit
// device-wide synchronisation cudaMalloc / cudaFree can cause.  woden_truncate_select keeps its ranked
// list in a context arena that grows with cudaMalloc; none of those callers can afford that call.
//
// What this file does instead: the ranked list lives in ONE fixed array that is part of the library
// image (`g_scratch` below, WODEN_STATIC_TRUNCATE_MAX entries, 192 KiB).  Every GPU that loads the
// library carries that array from module load until the process exits, whether or not this entry point
// is ever used.  No cudaMalloc, cudaFree, woden_create or other allocating call is made here.
//
// The kernels restate truncate.cu's three steps (rank by counting, one sequential running sum in FP64,
// keep flags) so that both entry points decide N_comp on identical numbers; the existing path is left
// as it is.
#include <cstdio>
#include <mutex>

#include "../../include/woden_b200.h"
#include "kernels.h"

namespace {

constexpr int MAX_N = WODEN_STATIC_TRUNCATE_MAX;
constexpr int MAX_DEVICES = 64;

// The scratch: |I_j| in ranked order, then the rank of every component.  In HOST code the name
// `g_scratch` is only a handle for the runtime's symbol table -- it is not a device address, and a
// kernel handed `&g_scratch` would fault (or quietly use host memory where the GPU can reach it).  Host
// code therefore asks the runtime for the real address once per device (scratch_for_current_device).
struct StaticScratch {
    double sorted[MAX_N];
    int rank[MAX_N];
};
static __device__ __align__(256) StaticScratch g_scratch;

std::mutex g_mu;
StaticScratch *g_dev_ptr[MAX_DEVICES] = {};      // device address of g_scratch on each device, once known
thread_local char g_msg[256] = "";

int fail(int status, const char *what, cudaError_t e = cudaSuccess)
{
    if (e != cudaSuccess) { snprintf(g_msg, sizeof g_msg, "%s: %s", what, cudaGetErrorString(e)); cudaGetLastError(); }
    else snprintf(g_msg, sizeof g_msg, "%s", what);
    return status;
}

// Set-up, once per device and with that device current: the device address of this device's copy of
// the array.  (Each device has its own copy; the address from one device must not be used on another.)
int scratch_for_current_device(StaticScratch **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(WODEN_ERR_CUDA, "cudaGetDevice", e);
    if (dev < 0 || dev >= MAX_DEVICES) return fail(WODEN_ERR_DIM, "device ordinal beyond the 64 this entry point tracks");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_dev_ptr[dev]) {
        StaticScratch *p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_scratch);
        if (e != cudaSuccess || !p) return fail(WODEN_ERR_CUDA, "cudaGetSymbolAddress(static truncation scratch)", e);
        g_dev_ptr[dev] = p;
    }
    *out = g_dev_ptr[dev];
    return WODEN_OK;
}

// as in truncate.cu: a non-finite weight ranks as 0 (there is no context here whose counter could report it)
__device__ __forceinline__ double static_abs(double w) { return isfinite(w) ? fabs(w) : 0.0; }

// rank_j = number of components with a larger |I| (equal values in their original order): Eq 24
__global__ void static_rank_kernel(const double *__restrict__ w, int n, StaticScratch *__restrict__ s)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const double a = static_abs(w[j]);
    int r = 0;
    for (int i = 0; i < n; ++i) {
        const double b = static_abs(w[i]);
        r += (b > a) || (b == a && i < j);
    }
    s->rank[j] = r;
    s->sorted[r] = a;
}

// Eq 23: the longest ranked prefix whose sum stays within f_comp * total, one thread, list order
__global__ void static_count_kernel(const StaticScratch *__restrict__ s, int n, double f_comp, int *__restrict__ n_keep)
{
    if (threadIdx.x || blockIdx.x) return;
    if (f_comp >= 1.0) { *n_keep = n; return; }
    double total = 0.0;
    for (int k = 0; k < n; ++k) total += s->sorted[k];
    const double limit = f_comp * total * (1.0 + 1e-15);
    double run = 0.0;
    int keep = 0;
    for (int k = 0; k < n; ++k) {
        run += s->sorted[k];
        if (run <= limit) keep = k + 1; else break;
    }
    *n_keep = keep;
}

__global__ void static_flag_kernel(const StaticScratch *__restrict__ s, int n, const int *__restrict__ n_keep,
                                   int *__restrict__ keep)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) keep[j] = s->rank[j] < *n_keep ? 1 : 0;
}

}  // namespace

extern "C" {

int woden_truncate_select_static(int n, const double *weights, double f_comp, int *keep, int *n_keep, void *cuda_stream)
{
    g_msg[0] = 0;
    if (n < 0 || !(f_comp >= 0.0)) return fail(WODEN_ERR_DIM, "n < 0 or f_comp not >= 0");
    if (n > MAX_N)
        return fail(WODEN_ERR_STATIC_LIMIT,
                    "n exceeds WODEN_STATIC_TRUNCATE_MAX (16384), the size of the built-in scratch array; "
                    "use woden_truncate_select, which allocates");
    if (!n_keep || (n > 0 && (!weights || !keep))) return fail(WODEN_ERR_NULL, "a required pointer is NULL");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t e;
    if (n == 0) {
        e = cudaMemsetAsync(n_keep, 0, sizeof(int), st);
        return e == cudaSuccess ? WODEN_OK : fail(WODEN_ERR_CUDA, "clear n_keep", e);
    }
    StaticScratch *s = nullptr;
    int rc = scratch_for_current_device(&s);
    if (rc != WODEN_OK) return rc;
    // the array still holds the previous call's ranked list: start this call's part of it from zero, so that
    // whatever the weights are, nothing of an earlier call can enter this call's running sum
    e = cudaMemsetAsync(s->sorted, 0, sizeof(double) * (size_t)n, st);
    if (e != cudaSuccess) return fail(WODEN_ERR_CUDA, "clear static scratch", e);
    static_rank_kernel<<<(n + 127) / 128, 128, 0, st>>>(weights, n, s); woden::note_launch();
    static_count_kernel<<<1, 32, 0, st>>>(s, n, f_comp, n_keep); woden::note_launch();
    static_flag_kernel<<<(n + 255) / 256, 256, 0, st>>>(s, n, n_keep, keep); woden::note_launch();
    e = cudaGetLastError();
    return e == cudaSuccess ? WODEN_OK : fail(WODEN_ERR_CUDA, "static truncation launch", e);
}

const char *woden_static_last_error(void) { return g_msg; }

}  // extern "C"
