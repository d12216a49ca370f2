// pipes.cu -- pipe-rate microbenchmarks that MEASURE the ALU roofline denominators on the B200
// the library runs on (MEASURED_PEAKS.json has no FP32 / MUFU / FP64 figure).
// Each kernel issues long runs of one instruction class over 16 independent register chains per
// thread, on every SM, and reports thread-operations per second plus the SM clock seen by
// clock64 against the global nanosecond timer.
#include <cstdint>
#include <cstdio>

#include "kernels.h"

namespace woden {
namespace {

constexpr int CHAINS = 16;
constexpr int PIPE_THREADS = 512;
constexpr int PIPE_CTAS_PER_SM = 2;

enum { P_FFMA = 0, P_MUFU = 1, P_DFMA = 2, P_I2F = 3, P_LOP3 = 4, P_FFMA2 = 5, P_FFMA_IMM = 6,
       P_F2F = 7, P_MUFU_EX2 = 8, P_MUFU_FFMA = 9, P_FFMA_3REG = 10, P_FFMA2_3REG = 11, P_FFMA2_BCAST = 12,
       P_FFMA2_UR = 13, P_WALK = 14, P_COUNT };

__constant__ unsigned long long PIPE_C[1024];     // uniform operands (values are irrelevant: zero)

__device__ __forceinline__ uint64_t globaltimer_ns()
{
    uint64_t t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

template <int WHICH>
__global__ void __launch_bounds__(PIPE_THREADS) pipe_kernel(int iters, float seed, float *sink,
                                                            unsigned long long *clk)
{
    float a[CHAINS];
    double d[CHAINS / 2];
    unsigned u[CHAINS];
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) {
        a[i] = seed + 0.001f * (threadIdx.x + i);
        u[i] = __float_as_uint(a[i]) + i;
    }
#pragma unroll
    for (int i = 0; i < CHAINS / 2; ++i) d[i] = (double)a[i];
    const float b = seed * 0.999f, c = seed * 1e-3f;
    const double db = (double)b, dc = (double)c;
    unsigned long long t0 = 0, c0 = 0;
    if (threadIdx.x == 0) { t0 = globaltimer_ns(); c0 = clock64(); }

    for (int it = 0; it < iters; ++it) {
        if (WHICH == P_FFMA) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < CHAINS; ++i) a[i] = fmaf(a[i], b, c);
        } else if (WHICH == P_FFMA_IMM) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < CHAINS; ++i) a[i] = fmaf(a[i], 0.99993f, 1.0e-3f);
        } else if (WHICH == P_FFMA2) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < CHAINS; i += 2) {
                    unsigned long long x, y, z;
                    asm("mov.b64 %0, {%1, %2};" : "=l"(x) : "f"(a[i]), "f"(a[i + 1]));
                    asm("mov.b64 %0, {%1, %2};" : "=l"(y) : "f"(b), "f"(b));
                    asm("mov.b64 %0, {%1, %2};" : "=l"(z) : "f"(c), "f"(c));
                    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(x) : "l"(x), "l"(y), "l"(z));
                    asm("mov.b64 {%0, %1}, %2;" : "=f"(a[i]), "=f"(a[i + 1]) : "l"(x));
                }
        } else if (WHICH == P_FFMA_3REG) {
            // three distinct register operands per FFMA (no operand shared between neighbours)
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < CHAINS; i += 2) {
                    a[i] = fmaf(a[i + 1], __uint_as_float(u[i]), a[i]);
                    a[i + 1] = fmaf(a[i], __uint_as_float(u[i + 1]), a[i + 1]);
                }
        } else if (WHICH == P_FFMA2_3REG) {
            // x = fma2(y, z, x) with three distinct 64-bit register pairs
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < CHAINS; i += 4) {
                    unsigned long long x, y, z, w2;
                    asm("mov.b64 %0, {%1, %2};" : "=l"(x) : "f"(a[i]), "f"(a[i + 1]));
                    asm("mov.b64 %0, {%1, %2};" : "=l"(y) : "f"(a[i + 2]), "f"(a[i + 3]));
                    asm("mov.b64 %0, {%1, %2};" : "=l"(z) : "r"(u[i]), "r"(u[i + 1]));
                    asm("mov.b64 %0, {%1, %2};" : "=l"(w2) : "r"(u[i + 2]), "r"(u[i + 3]));
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(x) : "l"(y), "l"(z));
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(y) : "l"(x), "l"(w2));
                    asm("mov.b64 {%0, %1}, %2;" : "=f"(a[i]), "=f"(a[i + 1]) : "l"(x));
                    asm("mov.b64 {%0, %1}, %2;" : "=f"(a[i + 2]), "=f"(a[i + 3]) : "l"(y));
                }
        } else if (WHICH == P_FFMA2_BCAST) {
            // x = fma2((c,c), y, x): scalar broadcast operand (SASS R.F32) + two distinct pairs
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < CHAINS; i += 4) {
                    unsigned long long x, y, cc;
                    asm("mov.b64 %0, {%1, %2};" : "=l"(x) : "f"(a[i]), "f"(a[i + 1]));
                    asm("mov.b64 %0, {%1, %2};" : "=l"(y) : "f"(a[i + 2]), "f"(a[i + 3]));
                    asm("mov.b64 %0, {%1, %2};" : "=l"(cc) : "f"(b), "f"(b));
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(x) : "l"(cc), "l"(y));
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(y) : "l"(cc), "l"(x));
                    asm("mov.b64 {%0, %1}, %2;" : "=f"(a[i]), "=f"(a[i + 1]) : "l"(x));
                    asm("mov.b64 {%0, %1}, %2;" : "=f"(a[i + 2]), "=f"(a[i + 3]) : "l"(y));
                }
        } else if (WHICH == P_FFMA2_UR) {
            // x = fma2(y, U, x): two changing register pairs + one uniform-register pair (constant bank)
            unsigned long long x[CHAINS / 4], y[CHAINS / 4];
#pragma unroll
            for (int i = 0; i < CHAINS / 4; ++i) {
                asm("mov.b64 %0, {%1, %2};" : "=l"(x[i]) : "f"(a[4 * i]), "f"(a[4 * i + 1]));
                asm("mov.b64 %0, {%1, %2};" : "=l"(y[i]) : "f"(a[4 * i + 2]), "f"(a[4 * i + 3]));
            }
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < CHAINS / 4; ++i) {
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(x[i]) : "l"(y[i]), "l"(PIPE_C[(it * 32 + r * 8 + 2 * i) & 1023]));
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(y[i]) : "l"(x[i]), "l"(PIPE_C[(it * 32 + r * 8 + 2 * i + 1) & 1023]));
                }
#pragma unroll
            for (int i = 0; i < CHAINS / 4; ++i) {
                asm("mov.b64 {%0, %1}, %2;" : "=f"(a[4 * i]), "=f"(a[4 * i + 1]) : "l"(x[i]));
                asm("mov.b64 {%0, %1}, %2;" : "=f"(a[4 * i + 2]), "=f"(a[4 * i + 3]) : "l"(y[i]));
            }
        } else if (WHICH == P_WALK) {
            // the channel-walking kernel's instruction pattern per channel pair (predict_walk.cu), two
            // independent chains: rn = c rc + ra; in = c ic + ia (scalar c); acc_re += U rc; acc_im += U ic
            unsigned long long rc[2], ic[2], ra[2], ia[2], ar[2], ai[2], cc;
            asm("mov.b64 %0, {%1, %2};" : "=l"(cc) : "f"(b), "f"(b));
#pragma unroll
            for (int d = 0; d < 2; ++d) {
                asm("mov.b64 %0, {%1, %2};" : "=l"(rc[d]) : "f"(a[8 * d]), "f"(a[8 * d + 1]));
                asm("mov.b64 %0, {%1, %2};" : "=l"(ic[d]) : "f"(a[8 * d + 2]), "f"(a[8 * d + 3]));
                asm("mov.b64 %0, {%1, %2};" : "=l"(ra[d]) : "f"(a[8 * d + 4]), "f"(a[8 * d + 5]));
                asm("mov.b64 %0, {%1, %2};" : "=l"(ia[d]) : "f"(a[8 * d + 6]), "f"(a[8 * d + 7]));
                asm("mov.b64 %0, {%1, %2};" : "=l"(ar[d]) : "r"(u[8 * d]), "r"(u[8 * d + 1]));
                asm("mov.b64 %0, {%1, %2};" : "=l"(ai[d]) : "r"(u[8 * d + 2]), "r"(u[8 * d + 3]));
            }
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int d = 0; d < 2; ++d) {
                    const unsigned long long U = PIPE_C[(it * 16 + r * 2 + d) & 1023];
                    unsigned long long rn, in;
                    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rn) : "l"(cc), "l"(rc[d]), "l"(ra[d]));
                    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(in) : "l"(cc), "l"(ic[d]), "l"(ia[d]));
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(ar[d]) : "l"(U), "l"(rc[d]));
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(ai[d]) : "l"(U), "l"(ic[d]));
                    ra[d] = rc[d]; ia[d] = ic[d]; rc[d] = rn; ic[d] = in;
                }
#pragma unroll
            for (int d = 0; d < 2; ++d) {
                asm("mov.b64 {%0, %1}, %2;" : "=f"(a[8 * d]), "=f"(a[8 * d + 1]) : "l"(rc[d]));
                asm("mov.b64 {%0, %1}, %2;" : "=f"(a[8 * d + 2]), "=f"(a[8 * d + 3]) : "l"(ic[d]));
                asm("mov.b64 {%0, %1}, %2;" : "=f"(a[8 * d + 4]), "=f"(a[8 * d + 5]) : "l"(ra[d]));
                asm("mov.b64 {%0, %1}, %2;" : "=f"(a[8 * d + 6]), "=f"(a[8 * d + 7]) : "l"(ia[d]));
                asm("mov.b64 {%0, %1}, %2;" : "=r"(u[8 * d]), "=r"(u[8 * d + 1]) : "l"(ar[d]));
                asm("mov.b64 {%0, %1}, %2;" : "=r"(u[8 * d + 2]), "=r"(u[8 * d + 3]) : "l"(ai[d]));
            }
        } else if (WHICH == P_MUFU) {
#pragma unroll
            for (int i = 0; i < CHAINS; i += 2) {
                a[i] = __sinf(a[i]);
                a[i + 1] = __cosf(a[i + 1]);
            }
        } else if (WHICH == P_MUFU_EX2) {
#pragma unroll
            for (int i = 0; i < CHAINS; ++i) asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(a[i]) : "f"(a[i]));
        } else if (WHICH == P_MUFU_FFMA) {
            // 2 MUFU + 12 FFMA per "eval": can the FMA pipe run under a saturated XU pipe?
#pragma unroll
            for (int i = 0; i < CHAINS; i += 8) {
                asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(a[i]) : "f"(a[i]));
                asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(a[i + 1]) : "f"(a[i + 1]));
#pragma unroll
                for (int r = 0; r < 2; ++r)
#pragma unroll
                    for (int k = 2; k < 8; ++k) a[i + k] = fmaf(a[i + k], b, c);
            }
        } else if (WHICH == P_DFMA) {
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int i = 0; i < CHAINS / 2; ++i) d[i] = fma(d[i], db, dc);
        } else if (WHICH == P_I2F) {
#pragma unroll
            for (int i = 0; i < CHAINS; ++i) u[i] = __float_as_uint((float)(int)u[i]) ^ 0x5a5a5a5u;
        } else if (WHICH == P_LOP3) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < CHAINS; ++i) u[i] = (u[i] & 0x007fffffu) | (u[(i + 1) % CHAINS] ^ 0x3f800000u);
        } else if (WHICH == P_F2F) {
#pragma unroll
            for (int i = 0; i < CHAINS / 2; ++i) d[i] = (double)((float)d[i]) + dc;
        }
    }

    if (threadIdx.x == 0) {
        unsigned long long c1 = clock64(), t1 = globaltimer_ns();
        if (blockIdx.x == 0) { clk[0] = c1 - c0; clk[1] = t1 - t0; }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) s += a[i] + __uint_as_float(u[i] & 0x3fffffffu);
#pragma unroll
    for (int i = 0; i < CHAINS / 2; ++i) s += (float)d[i];
    if (s == 123.456f) sink[0] = s;     // never true in practice; keeps the chains live
}

// thread-operations of the counted class per loop iteration per thread
double ops_per_iter(int which)
{
    switch (which) {
    case P_FFMA: case P_FFMA_IMM: case P_LOP3: return 4.0 * CHAINS;
    case P_FFMA2: case P_FFMA2_3REG: case P_FFMA2_BCAST: return 4.0 * CHAINS;   // scalar FMAs (2 per f32x2)
    case P_FFMA2_UR: return 4.0 * CHAINS;      // 4 x 8 FFMA2 = 64 scalar FMAs
    case P_WALK: return 8.0 * 2 * 4 * 2;       // 8 steps x 2 chains x 4 FFMA2 x 2 lanes
    case P_FFMA_3REG: return 4.0 * CHAINS;
    case P_MUFU: case P_MUFU_EX2: case P_I2F: return CHAINS;
    case P_MUFU_FFMA: return CHAINS / 8 * 2;    // MUFU ops; 12 FFMA ride along per 2 MUFU
    case P_DFMA: return CHAINS;                 // 2 x CHAINS/2
    case P_F2F: return CHAINS / 2;              // one F2F.F32.F64 (+ one F2F.F64.F32 + DADD) each
    }
    return 0.0;
}

template <int W>
cudaError_t run_one(int iters, int grid, float *sink, unsigned long long *clk, float *ms)
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    pipe_kernel<W><<<grid, PIPE_THREADS>>>(iters / 8 + 1, 1.0f, sink, clk); note_launch();     // warm-up
    cudaEventRecord(e0);
    pipe_kernel<W><<<grid, PIPE_THREADS>>>(iters, 1.0f, sink, clk); note_launch();
    cudaEventRecord(e1);
    cudaError_t err = cudaEventSynchronize(e1);
    if (err == cudaSuccess) err = cudaGetLastError();
    cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return err;
}

}  // namespace

cudaError_t run_pipe_rate(int which, int iters, double *thread_ops_per_s, double *sm_clock_hz)
{
    if (which < 0 || which >= P_COUNT || iters <= 0) return cudaErrorInvalidValue;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = sms * PIPE_CTAS_PER_SM;
    float *sink = nullptr;
    unsigned long long *clk = nullptr, hclk[2] = {0, 0};
    cudaError_t err = cudaMalloc(&sink, 16);
    if (err != cudaSuccess) return err;
    err = cudaMalloc(&clk, 16);
    if (err != cudaSuccess) { cudaFree(sink); return err; }
    float ms = 0.f;
    switch (which) {
    case P_FFMA: err = run_one<P_FFMA>(iters, grid, sink, clk, &ms); break;
    case P_MUFU: err = run_one<P_MUFU>(iters, grid, sink, clk, &ms); break;
    case P_DFMA: err = run_one<P_DFMA>(iters, grid, sink, clk, &ms); break;
    case P_I2F: err = run_one<P_I2F>(iters, grid, sink, clk, &ms); break;
    case P_LOP3: err = run_one<P_LOP3>(iters, grid, sink, clk, &ms); break;
    case P_FFMA2: err = run_one<P_FFMA2>(iters, grid, sink, clk, &ms); break;
    case P_FFMA_IMM: err = run_one<P_FFMA_IMM>(iters, grid, sink, clk, &ms); break;
    case P_F2F: err = run_one<P_F2F>(iters, grid, sink, clk, &ms); break;
    case P_MUFU_EX2: err = run_one<P_MUFU_EX2>(iters, grid, sink, clk, &ms); break;
    case P_MUFU_FFMA: err = run_one<P_MUFU_FFMA>(iters, grid, sink, clk, &ms); break;
    case P_FFMA_3REG: err = run_one<P_FFMA_3REG>(iters, grid, sink, clk, &ms); break;
    case P_FFMA2_3REG: err = run_one<P_FFMA2_3REG>(iters, grid, sink, clk, &ms); break;
    case P_FFMA2_BCAST: err = run_one<P_FFMA2_BCAST>(iters, grid, sink, clk, &ms); break;
    case P_FFMA2_UR: err = run_one<P_FFMA2_UR>(iters, grid, sink, clk, &ms); break;
    case P_WALK: err = run_one<P_WALK>(iters, grid, sink, clk, &ms); break;
    }
    if (err == cudaSuccess) err = cudaMemcpy(hclk, clk, 16, cudaMemcpyDeviceToHost);
    cudaFree(sink); cudaFree(clk);
    if (err != cudaSuccess) return err;
    const double total = ops_per_iter(which) * (double)iters * PIPE_THREADS * (double)grid;
    *thread_ops_per_s = total / (ms * 1e-3);
    *sm_clock_hz = hclk[1] ? (double)hclk[0] / ((double)hclk[1] * 1e-9) : 0.0;
    return cudaSuccess;
}

}  // namespace woden
