// act_quant.cu -- per-token absmax int8 activation quantiser, Eq. 4 lines 1-2.
//   alpha_m = fmaxf(absmax_m, 1e-5f) / 127.0f        true fp32 division (reading R1)
//   a_mj    = clamp(rint(x_mj / alpha_m), +-127)     true fp32 division, round-half-to-even (R1-R3)
// One CTA per row: the row is read with 128-bit loads into registers (up to 48 bf16 per thread),
// reduced to its absmax (warp shuffles + one smem hop), then quantised from the registers: one pass
// over HBM.  Rows longer than the register window are re-read (they hit L1/L2).
#include <cuda_bf16.h>
#include "common.cuh"
#include "quant.cuh"
#include "kernels.h"

namespace vla {


// One CTA of T threads per row, AQ_VMAX vectors of 8 bf16 per thread in registers.  Short rows use 64 threads so that
// more rows are in flight per SM; the kernel is bound by the two true divisions per element (~15 instructions).
template <int T, int AQ_VMAX>
__global__ void __launch_bounds__(T) act_quant_kernel(const uint4* __restrict__ x, int K, uint2* __restrict__ xq,
                                                      float* __restrict__ x_scale) {
    __shared__ float s_max[T / 32];
    pdl_wait();                                          // x may be the previous kernel's output
    const int row = blockIdx.x;
    const int nvec = K / 8;
    const uint4* xr = x + (size_t)row * nvec;
    uint2* qr = xq + (size_t)row * nvec;

    uint4 v[AQ_VMAX];
    float m = 0.0f;
#pragma unroll
    for (int i = 0; i < AQ_VMAX; ++i) {
        int idx = threadIdx.x + i * T;
        v[i] = (idx < nvec) ? xr[idx] : make_uint4(0, 0, 0, 0);
    }
#pragma unroll
    for (int i = 0; i < AQ_VMAX; ++i) m = absmax8(v[i], m);
    for (int idx = threadIdx.x + AQ_VMAX * T; idx < nvec; idx += T) m = absmax8(xr[idx], m);

#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
    if (T > 32) {
        if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = m;
        __syncthreads();
        m = s_max[0];
#pragma unroll
        for (int i = 1; i < T / 32; ++i) m = fmaxf(m, s_max[i]);
    }

    const float alpha = alpha_of(m);
    if (threadIdx.x == 0) x_scale[row] = alpha;
    pdl_launch_dependents();
#pragma unroll
    for (int i = 0; i < AQ_VMAX; ++i) {
        int idx = threadIdx.x + i * T;
        if (idx < nvec) qr[idx] = quant8(v[i], alpha);
    }
    for (int idx = threadIdx.x + AQ_VMAX * T; idx < nvec; idx += T) qr[idx] = quant8(xr[idx], alpha);
}

template <int T, int V>
static cudaError_t launch_aq(const void* x_bf16, int M, int K, int8_t* xq, float* x_scale, cudaStream_t s) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)M);
    cfg.blockDim = dim3(T);
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    count_launch();
    return cudaLaunchKernelEx(&cfg, act_quant_kernel<T, V>, (const uint4*)x_bf16, K, (uint2*)xq, x_scale);
}

cudaError_t launch_act_quant(const void* x_bf16, int M, int K, int8_t* xq, float* x_scale, cudaStream_t s) {
    // measured on B200 (M = 4096): K = 2560: 64 threads x 5 vectors 10.1 us vs 256 x 4 13.6 us; K = 8192: 256 x 4 wins
    // (at M = 544 the 256-thread form is the faster one: 2.9 vs 3.3 us -- few rows, latency-bound)
    if (K <= 8 * 5 * 64 && M >= 1024) return launch_aq<64, 5>(x_bf16, M, K, xq, x_scale, s);
    return launch_aq<256, 4>(x_bf16, M, K, xq, x_scale, s);
}

}  // namespace vla
