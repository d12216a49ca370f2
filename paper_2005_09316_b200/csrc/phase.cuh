// phase.cuh -- device helpers shared by the predict kernels: the FP64 -> FP32 phase hand-off
// without a conversion instruction (hard part H2), MUFU wrappers and the packed FP32x2
// arithmetic of sm_100 (fma/mul.rn.f32x2, SASS FFMA2 / FMUL2).
#pragma once
#include <cuda_runtime.h>

namespace woden {

constexpr double MAGIC23 = 805306368.0;  // 1.5 * 2^29 : ulp of the sum = 2^-23 turn
constexpr double MAGIC32 = 1572864.0;    // 1.5 * 2^20 : low word of the sum = frac as Q0.32
// Range of the two hand-offs.  phi + MAGIC23 stays in its binade while |phi| < 2^28 turns.  The
// Q0.32 form needs |phi| < 2^19 turns for MAGIC32 itself; with the magic constant 1.5*2^(20+k) the
// low word holds phi modulo 2^k turns in units of 2^(k-32) turn, and `<< k` leaves the fraction
// with k fewer bits -- at k = 9 the same 2^28 turns / 2^-23 turn as MAGIC23.
constexpr int PHASE_MAX_SHIFT = 9;
// smallest k with bound < 2^(19+k) (bound >= 0; returns > PHASE_MAX_SHIFT when out of range)
__device__ __forceinline__ int phase_shift_for(double bound)
{
    const int e = (__double2hiint(bound) >> 20) - 1023;         // floor(log2(bound)) for normal values
    return e >= 19 ? e - 18 : 0;
}
__device__ __forceinline__ double magic32_shifted(int k)
{
    return __hiloint2double(0x41380000 + (k << 20), 0);          // 1.5 * 2^(20 + k)
}
constexpr float TWO_PI_F = 6.283185307179586f;
constexpr float THREE_PI_F = 9.42477796076938f;
constexpr float Q32_TO_RAD = 1.4629180792671596e-09f;   // 2 pi / 2^32

// angle in [-pi, pi) equal to 2 pi (frac(phi) - 1/2), from r = phi + MAGIC23: the low mantissa
// word of r holds frac(phi) to 2^-23 turn; one LOP3 makes a float in [1,2), one FFMA the angle.
__device__ __forceinline__ float theta_from_magic(double r)
{
    const unsigned lo = (unsigned)__double2loint(r);
    const float x = __uint_as_float((lo & 0x007fffffu) | 0x3f800000u);   // 1 + frac(phi)
    return fmaf(x, TWO_PI_F, -THREE_PI_F);
}

// angle in [-pi, pi) equal to 2 pi frac(phi) (signed), from r = phi + MAGIC32
__device__ __forceinline__ float theta_from_q32(double r)
{
    return (float)__double2loint(r) * Q32_TO_RAD;
}

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- packed FP32x2: one instruction, two independent lanes ---------------------------------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

}  // namespace woden
