// lv_device.cuh -- device-side helpers shared by the kernel files of csrc/ (lv_kernels.cu,
// lv_force_tile.cu): the fp32 contract #1 expression, the approximate reciprocals of the
// pair force (reading R28), packed f32x2 arithmetic and the skin-list guard.
#pragma once

#include "lv_internal.cuh"

namespace {

constexpr unsigned kFull = 0xffffffffu;

template <int N> struct IntC { static constexpr int value = N; };

// Skin-list steps run the cell rebuild only when the device-side flag of this step is
// raised (LvDevState::rebuild); `guard` is null on every other path.
__device__ __forceinline__ bool skipped(const LvDevState *guard)
{
    return guard != nullptr && guard->rebuild[guard->step & 1] == 0u;
}

__device__ __forceinline__ int cell_coord(float x, float lo, float inv_h, int G)
{
    // fp32 contract #1: t = fl(fl(x - lo) * inv_h), clamp(floor t), NaN -> 0
    float t = __fmul_rn(__fsub_rn(x, lo), inv_h);
    float f = floorf(t);
    if (!(f >= 0.0f)) return 0;
    if (f > (float)(G - 1)) return G - 1;
    return (int)f;
}

__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Two fp32 lanes in one 64-bit register pair (sm_100 FADD2 / FMUL2 / FFMA2): each half is
// an IEEE round-to-nearest operation, so contract #2 holds per half; one instruction issue
// serves two candidates.
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
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// acc += a * b with the accumulator tied to one register pair (no copy at a loop back-edge)
__device__ __forceinline__ void fma2_acc(f32x2 &acc, f32x2 a, f32x2 b)
{
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}

}  // namespace
