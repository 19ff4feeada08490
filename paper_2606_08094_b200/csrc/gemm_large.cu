// gemm_large.cu -- large-M (prefill) ternary GEMM on the 5th-gen tensor cores, Eq. 4 line 3
// ("Packed weight tiles are decoded in shared memory; activation tiles are
// reused across outputs.  Products accumulate in 32-bit integers ...").
//
// One CTA computes a 128(channels) x TN(tokens) output tile:
//   MMA operand A = decoded weights  [128 ch  x 128 k] int8, K-major, SWIZZLE_128B  (written by decode warps)
//   MMA operand B = int8 activations [TN tok  x 128 k] int8, K-major, SWIZZLE_128B  (written by TMA)
//   D (TMEM)      = int32 [128 lanes = channels] x [TN columns = tokens]
// Warp roles (192 threads):
//   warp 0      TMA producer: cp.async.bulk of the 4 KiB packed weight tile + tensor-map load of the X tile
//   warp 1      TMEM allocator; one lane issues tcgen05.mma.cta_group::1.kind::i8 (4 x K=32 per k-block)
//   warps 2-5   decode: packed words (smem) -> int8 (64*q) -> swizzled A tile; fence.proxy.async; then,
//               after the last k-block, the epilogue: tcgen05.ld -> >>6 -> (float)acc*(alpha_m*beta) -> store
// Pipelines: full_w (TMA->decode), full_x (TMA->MMA), decoded (decode->MMA), empty (MMA commit->TMA).
#include <cuda.h>
#include <cuda_bf16.h>
#include "common.cuh"
#include "kernels.h"

namespace vla {

constexpr int LG_THREADS = 192;
constexpr int LG_STAGES = 4;
constexpr int LG_A_BYTES = TILE_N * TILE_K;             // 16384 decoded int8
constexpr int LG_X_BYTES = 256 * TILE_K;                // 32768 (TN <= 256)
constexpr int LG_W_BYTES = TILE_BYTES;                  // 4096 packed
constexpr int LG_SMEM = LG_STAGES * (LG_A_BYTES + LG_X_BYTES + LG_W_BYTES) + 1024 /*align*/ + 256 /*barriers*/;

__global__ void __launch_bounds__(LG_THREADS, 1) gemm_large_kernel(
    const __grid_constant__ CUtensorMap tmap_x, const uint8_t* __restrict__ packed,
    const float* __restrict__ w_scale, const float* x_scale, void* out,
    int M, int N, int K, int TN, int tmem_cols, int out_dtype) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* base_ptr = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t sA = base;                                           // [STAGES][16384]
    const uint32_t sX = sA + LG_STAGES * LG_A_BYTES;                    // [STAGES][32768]
    const uint32_t sW = sX + LG_STAGES * LG_X_BYTES;                    // [STAGES][4096]
    const uint32_t sBar = sW + LG_STAGES * LG_W_BYTES;
    uint8_t* pW = base_ptr + LG_STAGES * (LG_A_BYTES + LG_X_BYTES);
    uint8_t* pA = base_ptr;
    auto bar_full_w = [&](int s) { return sBar + 8u * s; };
    auto bar_full_x = [&](int s) { return sBar + 8u * (LG_STAGES + s); };
    auto bar_decoded = [&](int s) { return sBar + 8u * (2 * LG_STAGES + s); };
    auto bar_empty = [&](int s) { return sBar + 8u * (3 * LG_STAGES + s); };
    const uint32_t bar_acc = sBar + 8u * (4 * LG_STAGES);
    const uint32_t tmem_slot = sBar + 8u * (4 * LG_STAGES + 1);
    volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(base_ptr + (tmem_slot - base));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nb = blockIdx.x;                    // 128-channel tile
    const int m0 = blockIdx.y * TN;               // first token of this tile
    const int num_kb = K / TILE_K;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmap_x);
        for (int s = 0; s < LG_STAGES; ++s) {
            mbar_init(bar_full_w(s), 1);
            mbar_init(bar_full_x(s), 1);
            mbar_init(bar_decoded(s), 4);          // one arrive per decode warp
            mbar_init(bar_empty(s), 1);
        }
        mbar_init(bar_acc, 1);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_slot, (uint32_t)tmem_cols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        if (lane == 0) {
            const uint8_t* wsrc = packed + (size_t)nb * num_kb * TILE_BYTES;
            // weights do not depend on the previous kernel: prefetch the first stages before the PDL wait
            int pre = min(num_kb, LG_STAGES);
            for (int kb = 0; kb < pre; ++kb) {
                mbar_arrive_expect_tx(bar_full_w(kb), LG_W_BYTES);
                tma_bulk_g2s(sW + kb * LG_W_BYTES, wsrc + (size_t)kb * TILE_BYTES, LG_W_BYTES, bar_full_w(kb));
            }
            pdl_wait();
            for (int kb = 0; kb < num_kb; ++kb) {
                const int s = kb % LG_STAGES;
                const uint32_t ph = (kb / LG_STAGES) & 1;
                if (kb >= LG_STAGES) {
                    mbar_wait(bar_empty(s), ph ^ 1);
                    mbar_arrive_expect_tx(bar_full_w(s), LG_W_BYTES);
                    tma_bulk_g2s(sW + s * LG_W_BYTES, wsrc + (size_t)kb * TILE_BYTES, LG_W_BYTES, bar_full_w(s));
                }
                mbar_arrive_expect_tx(bar_full_x(s), (uint32_t)TN * TILE_K);
                tma_tensor2d_g2s(sX + s * LG_X_BYTES, &tmap_x, kb * TILE_K, m0, bar_full_x(s));
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            const uint32_t idesc = umma_idesc_i8(TILE_N, TN);
            for (int kb = 0; kb < num_kb; ++kb) {
                const int s = kb % LG_STAGES;
                const uint32_t ph = (kb / LG_STAGES) & 1;
                mbar_wait(bar_decoded(s), ph);
                mbar_wait(bar_full_x(s), ph);
                tc_fence_after();
                const uint64_t a_desc = umma_desc_k_sw128(sA + s * LG_A_BYTES);
                const uint64_t b_desc = umma_desc_k_sw128(sX + s * LG_X_BYTES);
#pragma unroll
                for (int k = 0; k < TILE_K / 32; ++k)
                    mma_i8_ss(tmem_base, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | k) != 0);
                mma_commit(bar_empty(s));
            }
            mma_commit(bar_acc);
        }
    } else {
        // ---------------- decode warps ----------------
        const int d = threadIdx.x - 64;
        const int t = d & 3, p = (d >> 2) & 1, q = (d >> 3) & 3, i32 = d >> 5;
        const int g = 2 * q + p;
        for (int kb = 0; kb < num_kb; ++kb) {
            const int s = kb % LG_STAGES;
            const uint32_t ph = (kb / LG_STAGES) & 1;
            mbar_wait(bar_full_w(s), ph);
            const uint8_t* wst = pW + s * LG_W_BYTES;
            uint8_t* ast = pA + s * LG_A_BYTES;
#pragma unroll
            for (int it = 0; it < 2; ++it) {
                const int h = p ^ it;
                const uint4 wv = *reinterpret_cast<const uint4*>(wst + ((i32 * 2 + h) * 32 + g * 4 + t) * 16);
                const uint32_t w4[4] = {wv.x, wv.y, wv.z, wv.w};
                const int pos = (4 * h + t) ^ g;              // SWIZZLE_128B: 16-byte chunk index ^ (row & 7)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint4 o = make_uint4(decode64<0>(w4[j]), decode64<1>(w4[j]), decode64<2>(w4[j]), decode64<3>(w4[j]));
                    *reinterpret_cast<uint4*>(ast + (i32 * 4 + j) * 1024 + g * 128 + pos * 16) = o;
                }
            }
            fence_proxy_async_smem();                         // generic-proxy stores -> visible to the tensor core
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_decoded(s));
        }
        // ---------------- epilogue ----------------
        mbar_wait(bar_acc, 0);
        tc_fence_after();
        const int lq = warp & 3;                              // TMEM lane quarter this warp may read
        const int ch = nb * TILE_N + lq * 32 + lane;
        const float beta = (out_dtype == 2) ? 0.0f : *w_scale;
        for (int c0 = 0; c0 < TN; c0 += 16) {
            if (m0 + c0 >= M) break;
            uint32_t r[16];
            tmem_ld_32x32b_x16(tmem_base + ((uint32_t)(lq * 32) << 16) + (uint32_t)c0, r);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                const int m = m0 + c0 + i;
                if (m < M) {
                    const int a = (int)r[i] >> 6;
                    const size_t o = (size_t)m * N + ch;
                    if (out_dtype == 2) {
                        reinterpret_cast<int*>(out)[o] = a;
                    } else {
                        const float y = dequant(a, __fmul_rn(x_scale[m], beta));
                        if (out_dtype == 0) reinterpret_cast<float*>(out)[o] = y;
                        else reinterpret_cast<__nv_bfloat16*>(out)[o] = __float2bfloat16_rn(y);
                    }
                }
            }
        }
    }
    pdl_launch_dependents();
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, (uint32_t)tmem_cols);
}

// ---------------------------------------------------------------- host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

static int pick_tn(int M) {
    int tiles = (M + 255) / 256;
    int tn = ((M + tiles - 1) / tiles + 15) / 16 * 16;
    return tn < 16 ? 16 : tn;
}

cudaError_t launch_gemm_large(const void* packed, const float* w_scale, const int8_t* xq, const float* x_scale,
                              int M, int N, int K, void* out, int out_dtype, cudaStream_t s) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return cudaErrorNotSupported;
    const int TN = pick_tn(M);
    int cols = 32;
    while (cols < TN) cols *= 2;

    CUtensorMap tm;
    cuuint64_t gdim[2] = {(cuuint64_t)K, (cuuint64_t)M};
    cuuint64_t gstr[1] = {(cuuint64_t)K};
    cuuint32_t box[2] = {(cuuint32_t)TILE_K, (cuuint32_t)TN};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, (void*)xq, gdim, gstr, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;

    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(gemm_large_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, LG_SMEM);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(N / TILE_N), (unsigned)((M + TN - 1) / TN));
    cfg.blockDim = dim3(LG_THREADS);
    cfg.dynamicSmemBytes = LG_SMEM;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    count_launch();
    return cudaLaunchKernelEx(&cfg, gemm_large_kernel, tm, (const uint8_t*)packed, w_scale, x_scale, out,
                              M, N, K, TN, cols, out_dtype);
}

// ---------------------------------------------------------------- INT8 tensor-pipe issue-rate probe
__global__ void __launch_bounds__(64, 1) i8_mma_probe_kernel(int iters) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* base_ptr = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t sA = base, sB = base + 16384, sBar = base + 16384 + 32768;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < (16384 + 32768) / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(base_ptr)[i] = 0x01010101u;
    fence_proxy_async_smem();
    if (threadIdx.x == 0) { mbar_init(sBar, 1); fence_barrier_init(); }
    if (warp == 1) tmem_alloc(sBar + 8, 256);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(base_ptr + 16384 + 32768 + 8);
    if (warp == 0 && lane == 0) {
        const uint32_t idesc = umma_idesc_i8(128, 256);
        const uint64_t a = umma_desc_k_sw128(sA), b = umma_desc_k_sw128(sB);
        for (int i = 0; i < iters; ++i) mma_i8_ss(tmem_base, a + 2 * (i & 3), b + 2 * (i & 3), idesc, i != 0);
        mma_commit(sBar);
        mbar_wait(sBar, 0);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, 256);
}

cudaError_t run_i8_mma_probe(int ctas, int mmas_per_cta, float* ms_out) {
    const int smem = 16384 + 32768 + 1024 + 64;
    cudaError_t e = cudaFuncSetAttribute(i8_mma_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    count_launch(2);
    i8_mma_probe_kernel<<<ctas, 64, smem>>>(mmas_per_cta);      // warm-up
    cudaEventRecord(a);
    i8_mma_probe_kernel<<<ctas, 64, smem>>>(mmas_per_cta);
    cudaEventRecord(b);
    e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) cudaEventElapsedTime(ms_out, a, b);
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    return e;
}

}  // namespace vla
