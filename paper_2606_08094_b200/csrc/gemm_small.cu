// gemm_small.cu -- small-M (action-chunk / decode) ternary GEMM, Eq. 4 line 3.
//
// Bandwidth-bound regime: the packed weights are streamed from HBM exactly once with one coalesced
// 128-bit load per lane (a 512-byte block = 32 channels x 64 k per warp), decoded in registers
// (2 ALU ops per 4 weights, common.cuh) and contracted against the int8 activations either on the
// integer ALUs (dp4a, VLA_PATH_SMALL_ALU -- the paper's "dp4a on CUDA cores" baseline instruction,
// P:L82) or on the warp-level int8 tensor-core MMA (mma.sync.m16n8k32, VLA_PATH_SMALL_TC -- the
// paper's IMMA instruction class), whose A fragments are exactly the four decoded words of a lane.
//
// Grid: (N/32) x KSPLIT CTAs of 8 warps.  A CTA owns 32 output channels and 1/KSPLIT of K; its warps
// stride over the 64-wide k blocks, keep int32 partial sums in registers, reduce them through shared
// memory, and -- when KSPLIT > 1 -- the KSPLIT CTAs of a thread-block cluster reduce over distributed
// shared memory into rank 0, which runs the fused dequant epilogue.  int32 sums are exact in any order.
// Weight loads are issued before griddepcontrol.wait so that under programmatic dependent launch the
// weight stream of call i+1 overlaps the tail of call i (weights never depend on the previous kernel).
#include <cooperative_groups.h>
#include <cuda_bf16.h>
#include "common.cuh"
#include "kernels.h"

namespace cg = cooperative_groups;

namespace vla {

constexpr int SM_WARPS = 8;
constexpr int SM_THREADS = SM_WARPS * 32;
constexpr int SM_UNROLL = 2;

// MTOK: padded token count (multiple of 8 for the MMA variant).
template <int MTOK, bool USE_MMA>
__global__ void __launch_bounds__(SM_THREADS) gemm_small_kernel(
    const uint8_t* __restrict__ packed, const float* __restrict__ w_scale, const int8_t* xq,
    const float* x_scale, int M, int N, int K, void* out, int out_dtype, int kq_per_cta, int ksplit) {
    __shared__ int red[SM_WARPS][MTOK][33];
    __shared__ int tile[MTOK][32];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, t = lane & 3;
    const int n32 = blockIdx.x;
    const int kq0 = blockIdx.y * kq_per_cta;
    const int kq1 = min(K / BLK_K, kq0 + kq_per_cta);

    constexpr int MT = USE_MMA ? MTOK / 8 : 1;
    int acc_mma[2][MT][4];
    int acc_alu[4][USE_MMA ? 1 : MTOK];
    if constexpr (USE_MMA) {
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int i = 0; i < 4; ++i) acc_mma[c][mt][i] = 0;
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int m = 0; m < MTOK; ++m) acc_alu[j][m] = 0;
    }

    bool first = true;
    for (int kq = kq0 + warp; kq < kq1 || first; kq += SM_WARPS * SM_UNROLL) {
        uint4 wv[SM_UNROLL];
#pragma unroll
        for (int u = 0; u < SM_UNROLL; ++u) {
            int kk = kq + u * SM_WARPS;
            wv[u] = (kk < kq1) ? ldg_nc_v4(packed + block_offset(n32, kk, K) + lane * 16) : make_uint4(0, 0, 0, 0);
        }
        if (first) { pdl_wait(); first = false; }       // activations come from the previous kernel
#pragma unroll
        for (int u = 0; u < SM_UNROLL; ++u) {
            const int kk = kq + u * SM_WARPS;
            if (kk >= kq1) continue;
            const uint32_t w4[4] = {wv[u].x, wv[u].y, wv[u].z, wv[u].w};
            const int8_t* xk = xq + (size_t)kk * BLK_K + t * 16;
            if constexpr (USE_MMA) {
                uint4 xv[MT];
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    int tok = mt * 8 + g;
                    xv[mt] = (tok < M) ? *reinterpret_cast<const uint4*>(xk + (size_t)tok * K) : make_uint4(0, 0, 0, 0);
                }
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const uint32_t wa = w4[2 * c], wb = w4[2 * c + 1];     // channels 16c+g and 16c+g+8
                    const uint32_t a0 = decode64<0>(wa), a1 = decode64<0>(wb), a2 = decode64<1>(wa), a3 = decode64<1>(wb);
                    const uint32_t e0 = decode64<2>(wa), e1 = decode64<2>(wb), e2 = decode64<3>(wa), e3 = decode64<3>(wb);
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        mma_m16n8k32_s8(acc_mma[c][mt], a0, a1, a2, a3, xv[mt].x, xv[mt].y);
                        mma_m16n8k32_s8(acc_mma[c][mt], e0, e1, e2, e3, xv[mt].z, xv[mt].w);
                    }
                }
            } else {
                uint32_t d[4][4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    d[j][0] = decode64<0>(w4[j]); d[j][1] = decode64<1>(w4[j]);
                    d[j][2] = decode64<2>(w4[j]); d[j][3] = decode64<3>(w4[j]);
                }
#pragma unroll
                for (int m = 0; m < MTOK; ++m) {
                    if (m < M) {
                        uint4 xv = *reinterpret_cast<const uint4*>(xk + (size_t)m * K);
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            int a = acc_alu[j][m];
                            a = __dp4a((int)d[j][0], (int)xv.x, a);
                            a = __dp4a((int)d[j][1], (int)xv.y, a);
                            a = __dp4a((int)d[j][2], (int)xv.z, a);
                            a = __dp4a((int)d[j][3], (int)xv.w, a);
                            acc_alu[j][m] = a;
                        }
                    }
                }
            }
        }
    }
    pdl_launch_dependents();

    // per-warp partials -> shared memory, red[warp][token][channel]
    if constexpr (USE_MMA) {
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                red[warp][mt * 8 + 2 * t][16 * c + g] = acc_mma[c][mt][0];
                red[warp][mt * 8 + 2 * t + 1][16 * c + g] = acc_mma[c][mt][1];
                red[warp][mt * 8 + 2 * t][16 * c + g + 8] = acc_mma[c][mt][2];
                red[warp][mt * 8 + 2 * t + 1][16 * c + g + 8] = acc_mma[c][mt][3];
            }
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int m = 0; m < MTOK; ++m) {
                int a = acc_alu[j][m];
                a += __shfl_xor_sync(0xFFFFFFFFu, a, 1);
                a += __shfl_xor_sync(0xFFFFFFFFu, a, 2);
                if ((m & 3) == t) red[warp][m][8 * j + g] = a;
            }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < MTOK * 32; idx += SM_THREADS) {
        int tok = idx >> 5, ch = idx & 31, s = 0;
#pragma unroll
        for (int w = 0; w < SM_WARPS; ++w) s += red[w][tok][ch];
        tile[tok][ch] = s;
    }

    if (ksplit > 1) {
        cg::cluster_group cluster = cg::this_cluster();
        cluster.sync();
        if (cluster.block_rank() == 0) {
            for (int idx = threadIdx.x; idx < MTOK * 32; idx += SM_THREADS) {
                int s = tile[idx >> 5][idx & 31];
                for (int r = 1; r < ksplit; ++r) s += cluster.map_shared_rank(&tile[0][0], r)[idx];
                tile[idx >> 5][idx & 31] = s;
            }
        }
        cluster.sync();                                   // peers may exit only after rank 0 has read them
        if (cluster.block_rank() != 0) return;
    } else {
        __syncthreads();
    }

    // fused dequant epilogue: y = (float)acc * (alpha_m * beta); the factor 64 of the decode is shifted out
    const float beta = (out_dtype == 2) ? 0.0f : *w_scale;
    const int n0 = n32 * BLK_N;
    for (int idx = threadIdx.x; idx < MTOK * 32; idx += SM_THREADS) {
        int tok = idx >> 5, ch = idx & 31;
        if (tok >= M) continue;
        int a = tile[tok][ch] >> 6;
        size_t o = (size_t)tok * N + n0 + ch;
        if (out_dtype == 2) {
            reinterpret_cast<int*>(out)[o] = a;
        } else {
            float y = dequant(a, __fmul_rn(x_scale[tok], beta));
            if (out_dtype == 0) reinterpret_cast<float*>(out)[o] = y;
            else reinterpret_cast<__nv_bfloat16*>(out)[o] = __float2bfloat16_rn(y);
        }
    }
}

template <int MTOK, bool USE_MMA>
static cudaError_t launch_one(const void* packed, const float* w_scale, const int8_t* xq, const float* x_scale,
                              int M, int N, int K, void* out, int out_dtype, cudaStream_t s) {
    const int n32 = N / BLK_N, kq = K / BLK_K;
    int ksplit = 1;
    while (n32 * ksplit < 296 && ksplit < 8 && kq / (ksplit * 2) >= 4) ksplit *= 2;
    const int kq_per_cta = (kq + ksplit - 1) / ksplit;

    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n32, (unsigned)ksplit);
    cfg.blockDim = dim3(SM_THREADS);
    cfg.stream = s;
    cudaLaunchAttribute at[2];
    int na = 0;
    at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
    if (ksplit > 1) {
        at[na].id = cudaLaunchAttributeClusterDimension;
        at[na].val.clusterDim.x = 1;
        at[na].val.clusterDim.y = (unsigned)ksplit;
        at[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = at;
    cfg.numAttrs = na;
    count_launch();
    return cudaLaunchKernelEx(&cfg, gemm_small_kernel<MTOK, USE_MMA>, (const uint8_t*)packed, w_scale, xq, x_scale,
                              M, N, K, out, out_dtype, kq_per_cta, ksplit);
}

cudaError_t launch_gemm_small(bool use_mma, const void* packed, const float* w_scale, const int8_t* xq,
                              const float* x_scale, int M, int N, int K, void* out, int out_dtype, cudaStream_t s) {
#define GO(MTOK, MMA) return launch_one<MTOK, MMA>(packed, w_scale, xq, x_scale, M, N, K, out, out_dtype, s)
    if (use_mma) {
        if (M <= 8) GO(8, true);
        if (M <= 16) GO(16, true);
        if (M <= 32) GO(32, true);
    } else {
        if (M <= 1) GO(1, false);
        if (M <= 2) GO(2, false);
        if (M <= 4) GO(4, false);
        if (M <= 8) GO(8, false);
        if (M <= 16) GO(16, false);
    }
#undef GO
    return cudaErrorInvalidValue;
}

}  // namespace vla
