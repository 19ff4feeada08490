// quant.cuh -- the activation quantiser's arithmetic, Eq. 4 lines 1-2, shared by
// act_quant.cu (stand-alone kernel) and gemm_program.cu (row-owner quant inside the persistent kernel).
//   alpha_m = fmaxf(absmax_m, 1e-5f) / 127.0f        true fp32 division (reading R1)
//   a_mj    = clamp(rint(x_mj / alpha_m), +-127)     true fp32 division, round-half-to-even (R1-R3)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace vla {

__device__ __forceinline__ float bf16lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }

__device__ __forceinline__ float absmax8(uint4 v, float m) {
    m = fmaxf(m, fabsf(bf16lo(v.x))); m = fmaxf(m, fabsf(bf16hi(v.x)));
    m = fmaxf(m, fabsf(bf16lo(v.y))); m = fmaxf(m, fabsf(bf16hi(v.y)));
    m = fmaxf(m, fabsf(bf16lo(v.z))); m = fmaxf(m, fabsf(bf16hi(v.z)));
    m = fmaxf(m, fabsf(bf16lo(v.w))); m = fmaxf(m, fabsf(bf16hi(v.w)));
    return m;
}

__device__ __forceinline__ uint32_t q1(float x, float alpha) {
    float t = __fdiv_rn(x, alpha);
    int r = __float2int_rn(t);                           // round-half-to-even
    r = max(-127, min(127, r));
    return (uint32_t)r & 0xFFu;
}

__device__ __forceinline__ uint2 quant8(uint4 v, float alpha) {
    uint2 o;
    o.x = q1(bf16lo(v.x), alpha) | (q1(bf16hi(v.x), alpha) << 8) | (q1(bf16lo(v.y), alpha) << 16) | (q1(bf16hi(v.y), alpha) << 24);
    o.y = q1(bf16lo(v.z), alpha) | (q1(bf16hi(v.z), alpha) << 8) | (q1(bf16lo(v.w), alpha) << 16) | (q1(bf16hi(v.w), alpha) << 24);
    return o;
}

__device__ __forceinline__ float alpha_of(float absmax) { return __fdiv_rn(fmaxf(absmax, 1e-5f), 127.0f); }

}  // namespace vla
