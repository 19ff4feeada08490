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

// ---------------------------------------------------------------- exact fast quantiser (program kernel)
// Exact shortcut for  a = rint(x / alpha)  (quant.cuh's q1, two true divisions):  with  inv = RN(1 / alpha),
// the products x * inv * (1 -+ 2^-19) bracket fl(x / alpha) (which is x / alpha within 2^-24 relative), and an FMA with
// 1.5 * 2^23 rounds each of them to the nearest integer, ties to even, exactly.  rint(fl(.)) is monotone, so when both
// ends give the same integer it IS the result; when they differ (a rounding boundary inside the bracket: < 5e-4 of the
// elements) the 16 elements are redone with the true-division quantiser.  |x / alpha| <= 127 (1 + 2^-23): no clamp.
// Two elements per instruction: fma.rn.f32x2.
__device__ __forceinline__ uint32_t quant4_fast(uint32_t u0, uint32_t u1, float2 ilo, float2 ihi, uint32_t& diff) {
    const float2 MAGIC = make_float2(12582912.0f, 12582912.0f);
    const float2 x01 = make_float2(bf16lo(u0), bf16hi(u0)), x23 = make_float2(bf16lo(u1), bf16hi(u1));
    const float2 a01 = __ffma2_rn(x01, ilo, MAGIC), b01 = __ffma2_rn(x01, ihi, MAGIC);
    const float2 a23 = __ffma2_rn(x23, ilo, MAGIC), b23 = __ffma2_rn(x23, ihi, MAGIC);
    const uint32_t a0 = __float_as_uint(a01.x), a1 = __float_as_uint(a01.y), a2 = __float_as_uint(a23.x), a3 = __float_as_uint(a23.y);
    diff |= (a0 ^ __float_as_uint(b01.x)) | (a1 ^ __float_as_uint(b01.y));
    diff |= (a2 ^ __float_as_uint(b23.x)) | (a3 ^ __float_as_uint(b23.y));
    // the int8 result is the low byte of each sum (0x4B400000 + r)
    return __byte_perm(__byte_perm(a0, a1, 0x0040), __byte_perm(a2, a3, 0x0040), 0x5410);
}
// Rare path (a rounding boundary inside an element's bracket): redo exactly those elements with the true-division
// quantiser of quant.cuh.  One out-of-line copy; the fast path is inlined per task.
__device__ __forceinline__ uint32_t patch2(uint32_t u, uint32_t o2, int shift, float4 sc) {
    const float MAGIC = 12582912.0f;
    const float x0 = bf16lo(u), x1 = bf16hi(u);
    if (__float_as_uint(__fmaf_rn(x0, sc.y, MAGIC)) != __float_as_uint(__fmaf_rn(x0, sc.z, MAGIC)))
        o2 = (o2 & ~(0xFFu << shift)) | (q1(x0, sc.x) << shift);
    if (__float_as_uint(__fmaf_rn(x1, sc.y, MAGIC)) != __float_as_uint(__fmaf_rn(x1, sc.z, MAGIC)))
        o2 = (o2 & ~(0xFF00u << shift)) | (q1(x1, sc.x) << (shift + 8));
    return o2;
}
static __device__ __noinline__ uint4 quant16_patch(uint4 a, uint4 b, float4 sc, uint4 o) {
    o.x = patch2(a.y, patch2(a.x, o.x, 0, sc), 16, sc);
    o.y = patch2(a.w, patch2(a.z, o.y, 0, sc), 16, sc);
    o.z = patch2(b.y, patch2(b.x, o.z, 0, sc), 16, sc);
    o.w = patch2(b.w, patch2(b.z, o.w, 0, sc), 16, sc);
    return o;
}
__device__ __forceinline__ uint4 quant16(uint4 a, uint4 b, float4 sc) {      // sc = {alpha, inv_lo, inv_hi, -}
    const float2 ilo = make_float2(sc.y, sc.y), ihi = make_float2(sc.z, sc.z);
    uint32_t diff = 0;
    uint4 o;
    o.x = quant4_fast(a.x, a.y, ilo, ihi, diff);
    o.y = quant4_fast(a.z, a.w, ilo, ihi, diff);
    o.z = quant4_fast(b.x, b.y, ilo, ihi, diff);
    o.w = quant4_fast(b.z, b.w, ilo, ihi, diff);
    if (diff != 0u) o = quant16_patch(a, b, sc, o);          // rare: a rounding boundary is too close
    return o;
}
// the same for one vector of 8 (stand-alone act_quant kernel)
static __device__ __noinline__ uint2 quant8_patch(uint4 a, float4 sc, uint2 o) {
    o.x = patch2(a.y, patch2(a.x, o.x, 0, sc), 16, sc);
    o.y = patch2(a.w, patch2(a.z, o.y, 0, sc), 16, sc);
    return o;
}
__device__ __forceinline__ uint2 quant8_fast(uint4 a, float4 sc) {
    const float2 ilo = make_float2(sc.y, sc.y), ihi = make_float2(sc.z, sc.z);
    uint32_t diff = 0;
    uint2 o;
    o.x = quant4_fast(a.x, a.y, ilo, ihi, diff);
    o.y = quant4_fast(a.z, a.w, ilo, ihi, diff);
    if (diff != 0u) o = quant8_patch(a, sc, o);
    return o;
}
// absmax of 8 bf16 as a packed pair of 15-bit magnitudes (bf16 magnitudes order like unsigned integers)
__device__ __forceinline__ uint32_t absmax8_packed(uint4 v, uint32_t m) {
    m = __vmaxu2(m, v.x & 0x7FFF7FFFu);
    m = __vmaxu2(m, v.y & 0x7FFF7FFFu);
    m = __vmaxu2(m, v.z & 0x7FFF7FFFu);
    m = __vmaxu2(m, v.w & 0x7FFF7FFFu);
    return m;
}

// the larger half of a packed absmax pair as fp32
__device__ __forceinline__ float absmax_unpack(uint32_t m) { return fmaxf(bf16lo(m), bf16hi(m)); }

// {alpha, 1/alpha * (1 - 2^-19), 1/alpha * (1 + 2^-19), -}
__device__ __forceinline__ float4 quant_scales_of_alpha(float alpha) {
    const float inv = __frcp_rn(alpha);
    return make_float4(alpha, __fmul_rn(inv, 1.0f - 1.9073486328125e-06f), __fmul_rn(inv, 1.0f + 1.9073486328125e-06f), 0.0f);
}

}  // namespace vla
