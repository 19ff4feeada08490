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

// ---------------------------------------------------------------- exact fast quantiser (persistent kernels)
// Exact shortcut for  a = rint(x / alpha)  (q1 above: two true divisions):  with  inv = RN(1 / alpha), the products
// x * inv * (1 -+ 2^-19) bracket fl(x / alpha) (which is x / alpha within 2^-24 relative), and an FMA with 1.5 * 2^23 rounds
// each of them to the nearest integer, ties to even, exactly.  rint(fl(.)) is monotone, so when both ends give the same
// integer it IS the result; when they differ (a rounding boundary inside the bracket) that ELEMENT is redone with q1.
// |x / alpha| <= 127 (1 + 2^-23): no clamp.  Two elements per instruction: fma.rn.f32x2.
// How often: on bf16 data ~1 % of all 8-element vectors have such an element (measured) -- with 8-bit mantissas x / alpha
// is often an exact rational tie k + 1/2 -- so almost every warp takes the rare branch for one or two lanes per round.  The
// branch therefore has to be SHORT: the low bytes of both bracket ends are packed (PRMT) and XORed, a non-zero byte marks
// the element, and only marked elements run q1 (~40 instructions).  (Re-scanning all elements of the vector with scalar
// FMAs, as the first version did, cost 1.5 us per stage of the large programs and 1.6 us per phase of the M=8 stack.)
__device__ __forceinline__ uint32_t quant4_fast(uint32_t u0, uint32_t u1, float2 ilo, float2 ihi, uint32_t& dw) {
    const float2 MAGIC = make_float2(12582912.0f, 12582912.0f);
    const float2 x01 = make_float2(bf16lo(u0), bf16hi(u0)), x23 = make_float2(bf16lo(u1), bf16hi(u1));
    const float2 a01 = __ffma2_rn(x01, ilo, MAGIC), b01 = __ffma2_rn(x01, ihi, MAGIC);
    const float2 a23 = __ffma2_rn(x23, ilo, MAGIC), b23 = __ffma2_rn(x23, ihi, MAGIC);
    // the int8 result is the low byte of each sum (0x4B400000 + r)
    const uint32_t wa = __byte_perm(__byte_perm(__float_as_uint(a01.x), __float_as_uint(a01.y), 0x0040),
                                    __byte_perm(__float_as_uint(a23.x), __float_as_uint(a23.y), 0x0040), 0x5410);
    const uint32_t wb = __byte_perm(__byte_perm(__float_as_uint(b01.x), __float_as_uint(b01.y), 0x0040),
                                    __byte_perm(__float_as_uint(b23.x), __float_as_uint(b23.y), 0x0040), 0x5410);
    dw = wa ^ wb;                                        // adjacent integers differ in their low byte
    return wa;
}
// redo the elements marked in dw (non-zero byte e = element e of {u0 lo, u0 hi, u1 lo, u1 hi}) with the true divisions
__device__ __forceinline__ uint32_t fix4(uint32_t w, uint32_t dw, uint32_t u0, uint32_t u1, float alpha) {
    while (dw != 0u) {
        const int e = (__ffs((int)dw) - 1) >> 3;
        const uint32_t u = (e & 2) ? u1 : u0;
        const float x = (e & 1) ? bf16hi(u) : bf16lo(u);
        const uint32_t m = 0xFFu << (8 * e);
        w = (w & ~m) | (q1(x, alpha) << (8 * e));
        dw &= ~m;
    }
    return w;
}
__device__ __forceinline__ uint4 quant16(uint4 a, uint4 b, float4 sc) {      // sc = {alpha, inv_lo, inv_hi, -}
    const float2 ilo = make_float2(sc.y, sc.y), ihi = make_float2(sc.z, sc.z);
    uint32_t d0, d1, d2, d3;
    uint4 o;
    o.x = quant4_fast(a.x, a.y, ilo, ihi, d0);
    o.y = quant4_fast(a.z, a.w, ilo, ihi, d1);
    o.z = quant4_fast(b.x, b.y, ilo, ihi, d2);
    o.w = quant4_fast(b.z, b.w, ilo, ihi, d3);
    if ((d0 | d1 | d2 | d3) != 0u) {                         // rare per lane, common per warp: keep it short
        o.x = fix4(o.x, d0, a.x, a.y, sc.x);
        o.y = fix4(o.y, d1, a.z, a.w, sc.x);
        o.z = fix4(o.z, d2, b.x, b.y, sc.x);
        o.w = fix4(o.w, d3, b.z, b.w, sc.x);
    }
    return o;
}
// the same for one vector of 8
__device__ __forceinline__ uint2 quant8_fast(uint4 a, float4 sc) {
    const float2 ilo = make_float2(sc.y, sc.y), ihi = make_float2(sc.z, sc.z);
    uint32_t d0, d1;
    uint2 o;
    o.x = quant4_fast(a.x, a.y, ilo, ihi, d0);
    o.y = quant4_fast(a.z, a.w, ilo, ihi, d1);
    if ((d0 | d1) != 0u) {
        o.x = fix4(o.x, d0, a.x, a.y, sc.x);
        o.y = fix4(o.y, d1, a.z, a.w, sc.x);
    }
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
// A power-of-two alpha (absmax = 127 * 2^j: one bf16 mantissa in 128, so ~1 % of all rows) makes x / alpha EXACT, and with
// 8-bit bf16 mantissas a large share of its elements are exact ties k + 1/2, which a bracket of non-zero width can never
// decide: every vector of such a row would take the slow patch (measured: 2 % of all vectors, 1.5 us per stage).  There
// 1 / alpha is exact too, so x * (1/alpha) + MAGIC rounds the exact quotient, ties to even: the bracket collapses to a point.
__device__ __forceinline__ float4 quant_scales_of_alpha(float alpha) {
    const float inv = __frcp_rn(alpha);
    const bool dyadic = (__float_as_uint(alpha) & 0x007FFFFFu) == 0u;
    return make_float4(alpha, dyadic ? inv : __fmul_rn(inv, 1.0f - 1.9073486328125e-06f),
                       dyadic ? inv : __fmul_rn(inv, 1.0f + 1.9073486328125e-06f), 0.0f);
}

}  // namespace vla
