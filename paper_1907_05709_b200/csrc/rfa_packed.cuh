// rfa_packed.cuh -- two-voxels-per-instruction fp32 helpers (add.rn.f32x2 / fma.rn.f32x2 -> SASS FADD2 / FFMA2, which round
// per lane exactly like the scalar forms) and the fp16 residual packing, shared by the stepping kernels of librfa.so.
#pragma once
#include <cuda_fp16.h>

#include "rfa_device.cuh"

typedef unsigned long long u64;
__device__ __forceinline__ u64 pk(float lo, float hi)
{
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk(u64 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 add2(u64 a, u64 b)
{
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c)
{
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ float max3abs(float a, float b, float c) { return fmaxf(fmaxf(fabsf(a), fabsf(b)), fabsf(c)); }
__device__ __forceinline__ float max_abs4(const float4 v, float m) { return fmaxf(max3abs(v.x, v.y, v.z), fmaxf(fabsf(v.w), m)); }
__device__ __forceinline__ uint2 pack_h4(float a, float b, float c, float d)
{
    const __half2 lo = __floats2half2_rn(a, b), hi = __floats2half2_rn(c, d);
    uint2 r;
    r.x = *reinterpret_cast<const unsigned *>(&lo);
    r.y = *reinterpret_cast<const unsigned *>(&hi);
    return r;
}
__device__ __forceinline__ float4 unpack_h4(const uint2 v)
{
    const float2 lo = __half22float2(*reinterpret_cast<const __half2 *>(&v.x));
    const float2 hi = __half22float2(*reinterpret_cast<const __half2 *>(&v.y));
    return make_float4(lo.x, lo.y, hi.x, hi.y);
}

