// gemm_large.cu -- large-M (prefill) ternary GEMM on the 5th-gen tensor cores, Eq. 4 line 3
// ("Packed weight tiles are decoded in shared memory; activation tiles are
// reused across outputs.  Products accumulate in 32-bit integers ...").
//
// Persistent kernel: one CTA per SM walks the output tiles  t = blockIdx.x, += gridDim.x.
// A tile is 128 (channels) x TN (tokens, multiple of 16, <= 256):
//   MMA operand A = decoded weights  [128 ch  x 128 k] int8, K-major, SWIZZLE_128B  (written by the decode warps)
//   MMA operand B = int8 activations [TN tok  x 128 k] int8, K-major, SWIZZLE_128B  (written by TMA)
//   D (TMEM)      = int32 [128 lanes = channels] x [TN columns = tokens], TWO buffers (columns 0.. and 256..)
// Warp roles (15 warps):
//   warp 0       W producer: cp.async.bulk of the four 32-channel pieces of the packed weight tile per pipeline stage, KS KiB
//                each (the k blocks of a piece are contiguous; 1 KiB copies cap the chip at 3.7 TB/s = 0.164 us per k block
//                per SM, above the MMA time of narrow tiles), 6-deep ring (weights never depend on the previous kernel, so
//                this starts before griddepcontrol.wait)
//   warp 1       X producer: tensor-map (TMA) load of the [TN x 128] activation tile per k block, 4-deep ring
//   warp 2       TMEM allocator; one lane issues tcgen05.mma.cta_group::1.kind::i8 (4 x K=32 per k block)
//   warps 3-10   decode: packed words (smem) -> int8 (64*q) -> swizzled A tile (3-deep ring); fence.proxy.async
//   warps 11-14  epilogue: tcgen05.ld -> >>6 -> (float)acc*(alpha_m*beta) -> store, overlapped with the next
//                tile's main loop through the second TMEM buffer
#include <cuda.h>
#include <cuda_bf16.h>
#include "common.cuh"
#include "gemm_large.cuh"
#include "kernels.h"

namespace vla {

// KS = k blocks (of 128) per pipeline stage: 2 for token tiles <= 160 (eight MMAs per full/empty handoff), else 1.
template <int KS>
__global__ void __launch_bounds__(LG_THREADS, 1) gemm_large_kernel(
    const __grid_constant__ CUtensorMap tmap_x, const __grid_constant__ LgGroup grp,
    const float* __restrict__ x_scale, int M, int K, int TN, int NS, int NSW) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* base_ptr = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t x_tile = ((uint32_t)TN * TILE_K + 1023u) & ~1023u;
    const uint32_t stride = KS * (LG_A_BYTES + x_tile);               // [A x KS | X x KS]
    constexpr uint32_t X_OFF = KS * LG_A_BYTES;
    constexpr uint32_t W_STAGE = KS * LG_W_BYTES;
    const uint32_t sS = base;                                           // [NS]{A 16384 | X TN*128}
    const uint32_t sW = sS + (uint32_t)NS * stride;                     // [SW][4096]
    const uint32_t nsw = (uint32_t)NSW;                                 // packed-weight stages in use (<= LG_SW)
    const uint32_t sBar = sW + nsw * W_STAGE + LG_SCALE_BYTES;
    uint8_t* pS = base_ptr;
    uint8_t* pW = base_ptr + (size_t)NS * stride;
    float* pScale = reinterpret_cast<float*>(pW + nsw * W_STAGE);
    auto bar_full_w = [&](uint32_t s) { return sBar + 8u * s; };
    auto bar_empty_w = [&](uint32_t s) { return sBar + 8u * (LG_SW + s); };
    auto bar_full = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + s); };                  // A decoded + X landed
    auto bar_empty = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + LG_NS_MAX + s); };     // MMAs of the stage done
    auto bar_acc_full = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + 2 * LG_NS_MAX + s); };
    auto bar_acc_empty = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + 2 * LG_NS_MAX + 2 + s); };
    const uint32_t tmem_slot = sBar + 8u * LG_NBAR;
    volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(base_ptr + (tmem_slot - base));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int num_kb = K / TILE_K;
    const int tiles_n = grp.ct_begin[grp.n], tiles_m = (M + TN - 1) / TN;      // channel tiles over all linears of the group
    const int ntiles = tiles_n * tiles_m;
    const uint32_t ns = (uint32_t)NS;

    if (threadIdx.x == 0) {
        tma_prefetch_desc(&tmap_x);
        for (int s = 0; s < LG_SW; ++s) { mbar_init(bar_full_w(s), 1); mbar_init(bar_empty_w(s), 4); }
        for (int s = 0; s < LG_NS_MAX; ++s) { mbar_init(bar_full(s), 5); mbar_init(bar_empty(s), 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(bar_acc_full(s), 1); mbar_init(bar_acc_empty(s), 4); }
        fence_barrier_init();
    }
    if (warp == 2) tmem_alloc(tmem_slot, 512u);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    // Let the next kernel on the stream be scheduled NOW: its CTAs take an SM as soon as one of ours exits and run their
    // prologue (weight prefetch, decode of the first stages) under our tail; its own griddepcontrol.wait still waits for
    // this whole grid and its memory.
    pdl_launch_dependents();

    if (warp == 0) {
        // ---------------- W producer ----------------
        // a 128 x 128 tile is four 1 KiB pieces (one per 32-channel group), 8*K bytes apart: lanes 0-3 copy one each
        if (lane < 4) {                                       // one copy per 32-channel piece: its KS k blocks are contiguous
            const int piece = lane;
            uint32_t it = 0;
            RingCur cw;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const int ct = tile % tiles_n;
                int li = 0;
                for (int j = 1; j < grp.n; ++j) if (ct >= grp.ct_begin[j]) li = j;
                const int nb = ct - grp.ct_begin[li];
                const uint8_t* wsrc = grp.packed[li] + (size_t)(nb * 4 + piece) * num_kb * 1024;
                for (int kb = 0; kb < num_kb; kb += KS, ++it, cw.next(nsw)) {
                    const uint32_t s = cw.s;
                    if (cw.wrapped) mbar_wait(bar_empty_w(s), cw.ph ^ 1u);
                    if (lane == 0) mbar_arrive_expect_tx(bar_full_w(s), W_STAGE);
                    __syncwarp(0xFu);
                    tma_bulk_g2s(sW + s * W_STAGE + piece * (KS * 1024), wsrc + (size_t)kb * 1024, KS * 1024, bar_full_w(s));
                }
            }
        }
    } else if (warp == 1) {
        // ---------------- X producer ----------------
        if (lane == 0) {
            pdl_wait();                                       // activations come from the previous kernel
            uint32_t it = 0;
            RingCur cx;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const int m0 = (tile / tiles_n) * TN;
                for (int kb = 0; kb < num_kb; kb += KS, ++it, cx.next(ns)) {
                    const uint32_t s = cx.s;
                    if (cx.wrapped) mbar_wait(bar_empty(s), cx.ph ^ 1u);
                    mbar_arrive_expect_tx(bar_full(s), (uint32_t)KS * TN * TILE_K);
#pragma unroll
                    for (int kk = 0; kk < KS; ++kk)
                        tma_tensor2d_g2s(sS + s * stride + X_OFF + kk * x_tile, &tmap_x, (kb + kk) * TILE_K, m0, bar_full(s));
                }
            }
        }
    } else if (warp == 2) {
        // ---------------- MMA issuer: one wait, four MMAs, one commit per k block ----------------
        if (lane == 0) {
            const uint32_t idesc = umma_idesc_i8(TILE_N, TN);
            const uint64_t desc0 = umma_desc_k_sw128(sS);
            uint32_t it = 0, ti = 0;
            RingCur cm;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++ti) {
                const uint32_t ab = ti & 1;
                if (ti >= 2) mbar_wait(bar_acc_empty(ab), ((ti >> 1) & 1) ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + ab * 256u;
                for (int kb = 0; kb < num_kb; kb += KS, ++it, cm.next(ns)) {
                    const uint32_t s = cm.s;
                    mbar_wait(bar_full(s), cm.ph);
                    tc_fence_after();
#pragma unroll
                    for (int kk = 0; kk < KS; ++kk) {
                        // (descriptor = constant fields + (shared address >> 4): only the address part moves)
                        const uint64_t a_desc = desc0 + ((s * stride + kk * LG_A_BYTES) >> 4);
                        const uint64_t b_desc = desc0 + ((s * stride + X_OFF + kk * x_tile) >> 4);
#pragma unroll
                        for (int k = 0; k < TILE_K / 32; ++k)
                            mma_i8_ss(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | kk | k) != 0);
                    }
                    mma_commit(bar_empty(s));
                }
                mma_commit(bar_acc_full(ab));
            }
        }
    } else if (warp <= 10) {
        // ---------------- decode warps: two groups of four warps take alternate k blocks ----------------
        const int dgrp = (warp - 3) >> 2;
        const int d = (threadIdx.x - 96) & 127;
        const int t = d & 3, p = (d >> 2) & 1, q = (d >> 3) & 3, i32 = d >> 5;
        const int g = 2 * q + p;
        uint32_t it = 0;
            RingCur cd, cdw;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            for (int kb = 0; kb < num_kb; kb += KS, ++it, cd.next(ns), cdw.next(nsw)) {
                if ((int)(it & 1u) != dgrp) continue;
                const uint32_t sw = cdw.s, s = cd.s;
                mbar_wait(bar_full_w(sw), cdw.ph);
                const uint8_t* wst = pW + sw * W_STAGE;
                uint4 wv[KS][2];
#pragma unroll
                for (int kk = 0; kk < KS; ++kk)
#pragma unroll
                    for (int itx = 0; itx < 2; ++itx)
                        wv[kk][itx] = *reinterpret_cast<const uint4*>(wst + i32 * (KS * 1024) + kk * 1024 + ((p ^ itx) * 32 + g * 4 + t) * 16);
                if (cd.wrapped) mbar_wait(bar_empty(s), cd.ph ^ 1u);
#pragma unroll
                for (int kk = 0; kk < KS; ++kk) {
                    uint8_t* ast = pS + s * stride + kk * LG_A_BYTES;
#pragma unroll
                    for (int itx = 0; itx < 2; ++itx) {
                        const int h = p ^ itx;
                        const uint32_t w4[4] = {wv[kk][itx].x, wv[kk][itx].y, wv[kk][itx].z, wv[kk][itx].w};
                        const int pos = (4 * h + t) ^ g;      // SWIZZLE_128B: 16-byte chunk index ^ (row & 7)
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            uint4 o = make_uint4(decode64<0>(w4[j]), decode64<1>(w4[j]), decode64<2>(w4[j]), decode64<3>(w4[j]));
                            *reinterpret_cast<uint4*>(ast + (i32 * 4 + j) * 1024 + g * 128 + pos * 16) = o;
                        }
                    }
                }
                fence_proxy_async_smem();                     // generic-proxy stores -> visible to the tensor core
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(bar_empty_w(sw));
                    mbar_arrive(bar_full(s));
                }
            }
        }
    } else {
        // ---------------- epilogue warps ----------------
        const int lq = warp & 3;                              // TMEM lane quarter this warp may read
        float* sc = pScale + lq * 256;                        // this warp's alpha_m * beta of the tile's tokens
        const uint32_t sc_addr = sW + nsw * W_STAGE + (uint32_t)lq * 1024u;
        pdl_wait();                                           // x_scale comes from the previous kernel
        uint32_t ti = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++ti) {
            const int ct = tile % tiles_n, m0 = (tile / tiles_n) * TN;
            int li = 0;
            for (int j = 1; j < grp.n; ++j) if (ct >= grp.ct_begin[j]) li = j;
            const int nb = ct - grp.ct_begin[li], N = grp.N[li], out_dtype = grp.dtype[li];
            void* __restrict__ out = grp.out[li];
            const float beta = (out_dtype == 2) ? 0.0f : *grp.beta[li];
            const uint32_t ab = ti & 1;
            const int ch = nb * TILE_N + lq * 32 + lane;
            if (out_dtype != 2)
                for (int i = lane; i < TN; i += 32) sc[i] = (m0 + i < M) ? __fmul_rn(x_scale[m0 + i], beta) : 0.0f;
            __syncwarp();
            mbar_wait(bar_acc_full(ab), (ti >> 1) & 1);
            tc_fence_after();
            const uint32_t t_addr = tmem_base + ab * 256u + ((uint32_t)(lq * 32) << 16);
            for (int c0 = 0; c0 < TN; c0 += 16) {
                if (m0 + c0 >= M) break;
                uint32_t r[16];
                tmem_ld_32x32b_x16(t_addr + (uint32_t)c0, r);
                tmem_ld_wait();
                const int nrow = min(16, M - m0 - c0);
                float sv[16];                                 // explicit ld.shared: cannot alias the stores below
#pragma unroll
                for (int i4 = 0; i4 < 4; ++i4) {
                    const uint4 q4 = lds128_nv(sc_addr + (uint32_t)(c0 + 4 * i4) * 4u);
                    sv[4 * i4] = __uint_as_float(q4.x); sv[4 * i4 + 1] = __uint_as_float(q4.y);
                    sv[4 * i4 + 2] = __uint_as_float(q4.z); sv[4 * i4 + 3] = __uint_as_float(q4.w);
                }
                int acc[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) acc[i] = (int)r[i] >> 6;       // the decode's factor 64 leaves exactly
                const size_t o0 = (size_t)(m0 + c0) * N + ch;
                if (nrow == 16) {                              // full chunk: branch-free, 16 independent stores
                    if (out_dtype == 0) {
                        float* o = reinterpret_cast<float*>(out) + o0;
#pragma unroll
                        for (int i = 0; i < 16; ++i) o[(size_t)i * N] = dequant(acc[i], sv[i]);
                    } else if (out_dtype == 1) {
                        __nv_bfloat16* o = reinterpret_cast<__nv_bfloat16*>(out) + o0;
#pragma unroll
                        for (int i = 0; i < 16; ++i) o[(size_t)i * N] = __float2bfloat16_rn(dequant(acc[i], sv[i]));
                    } else {
                        int* o = reinterpret_cast<int*>(out) + o0;
#pragma unroll
                        for (int i = 0; i < 16; ++i) o[(size_t)i * N] = acc[i];
                    }
                } else {                                       // ragged tail of M
                    for (int i = 0; i < nrow; ++i) {
                        const size_t o = o0 + (size_t)i * N;
                        int a = 0; float sc_i = 0.0f;
#pragma unroll
                        for (int j = 0; j < 16; ++j) if (j == i) { a = acc[j]; sc_i = sv[j]; }
                        if (out_dtype == 0) reinterpret_cast<float*>(out)[o] = dequant(a, sc_i);
                        else if (out_dtype == 1) reinterpret_cast<__nv_bfloat16*>(out)[o] = __float2bfloat16_rn(dequant(a, sc_i));
                        else reinterpret_cast<int*>(out)[o] = a;
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_acc_empty(ab));    // this TMEM buffer may be overwritten
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc(tmem_base, 512u);
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

// Token-tile width TN (multiple of 16, <= 256) for a persistent grid of `sms` CTAs: minimise
//   waves * (cycles per k block), waves = ceil(tiles / sms).
// Measured on B200 (profiles/): a k block costs ~540 cycles at TN = 96 and ~610 at TN = 256 -- the shared-memory
// traffic of decode + operand fetch dominates, not the 2*TN cycles of the MMAs -- so cycles ~ 500 + 0.42*TN.
// Ties go to the wider tile (fewer re-decodes of the same weights).
int lg_pick_tn(int M, int N, int sms, bool k_even) {
    int best = 16;
    double best_cost = 1e30;
    for (int tn = 16; tn <= 256; tn += 16) {
        const int tiles_m = (M + tn - 1) / tn;
        if (tn > 16 && (tiles_m * (tn - 16) >= M)) continue;          // a narrower tile covers M with the same count
        const long tiles = (long)tiles_m * (N / TILE_N);
        const long waves = (tiles + sms - 1) / sms;
        // narrow tiles run two k blocks per stage (KS = 2): 0.21 us = ~410 cycles per k block at TN = 96
        const double per_kb = ((tn <= 112 && k_even) ? 370.0 : (tn <= 160 && k_even) ? 440.0 : 500.0) + 0.42 * tn;
        const double cost = (double)waves * per_kb;
        if (cost <= best_cost) { best_cost = cost; best = tn; }
    }
    return best;
}

// tensor map of the int8 activations xq [M,K]: box = [128 k, TN tokens], SWIZZLE_128B (operand B of the MMA)
cudaError_t lg_encode_x_map(void* tmap_out, const int8_t* xq, int M, int K, int TN) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return cudaErrorNotSupported;
    cuuint64_t gdim[2] = {(cuuint64_t)K, (cuuint64_t)M};
    cuuint64_t gstr[1] = {(cuuint64_t)K};
    cuuint32_t box[2] = {(cuuint32_t)TILE_K, (cuuint32_t)TN};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(reinterpret_cast<CUtensorMap*>(tmap_out), CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, (void*)xq, gdim, gstr, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t launch_gemm_large_grouped(const LgGroup& g, const int8_t* xq, const float* x_scale, int M, int K,
                                      cudaStream_t s) {
    const int N = g.ct_begin[g.n] * TILE_N;                  // all channels of the group
    int dev = 0, sms = 0;                                    // per call: a process may drive several devices
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
        return cudaErrorInvalidDevice;
    const int TN = lg_pick_tn(M, N, sms, (K / TILE_K) % 2 == 0);
    CUtensorMap tm;
    {
        const cudaError_t e = lg_encode_x_map(&tm, xq, M, K, TN);
        if (e != cudaSuccess) return e;
    }

    {   // function attributes are per device: set on every launch (cheap), no process-wide cache
        cudaError_t e = cudaFuncSetAttribute(gemm_large_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, LG_SMEM_LIMIT);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_large_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, LG_SMEM_LIMIT);
        if (e != cudaSuccess) return e;
    }
    const int ntiles = (N / TILE_N) * ((M + TN - 1) / TN);
    // narrow token tiles: two k blocks per stage (the MMAs of a 128 x TN x 32 step have a 31 ns floor for TN <= 112,
    // so four of them do not cover one full/empty handoff; eight do)
    const int KS = lg_pick_ks(TN, K);
    const int stage = KS * (int)lg_stage_stride(TN);
    // pipeline stages NS and packed-weight stages NSW from the shared memory there is: as many {A, X} stages as fit beside a
    // 6-deep weight ring, one more if a 4-deep ring makes room for it (TN = 112 with two k blocks per stage: 3, not 2).  The
    // ring depth stays EVEN: the two decode groups alternate over its stages, and with an odd depth a group would come back to a
    // stage last filled for the OTHER group, whose copy may not have landed yet -- its parity wait would fall through.
    int NS = 0, NSW = LG_SW;
    for (int nsw = LG_SW; nsw >= 4; nsw -= 2) {
        int ns = (LG_SMEM_LIMIT - (LG_SCALE_BYTES + 1024 + 8 * LG_NBAR + 16) - nsw * KS * LG_W_BYTES) / stage;
        if (ns > LG_NS_MAX) ns = LG_NS_MAX;
        if (ns > NS) { NS = ns; NSW = nsw; }
    }
    const int smem = NS * stage + NSW * KS * LG_W_BYTES + LG_SCALE_BYTES + 1024 + 8 * LG_NBAR + 16;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(ntiles < sms ? ntiles : sms));
    cfg.blockDim = dim3(LG_THREADS);
    cfg.dynamicSmemBytes = (size_t)smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    count_launch();
    if (KS == 2) return cudaLaunchKernelEx(&cfg, gemm_large_kernel<2>, tm, g, x_scale, M, K, TN, NS, NSW);
    return cudaLaunchKernelEx(&cfg, gemm_large_kernel<1>, tm, g, x_scale, M, K, TN, NS, NSW);
}

cudaError_t launch_gemm_large(const void* packed, const float* w_scale, const int8_t* xq, const float* x_scale,
                              int M, int N, int K, void* out, int out_dtype, cudaStream_t s) {
    LgGroup g = {};
    g.packed[0] = (const uint8_t*)packed;
    g.beta[0] = w_scale;
    g.out[0] = out;
    g.N[0] = N;
    g.dtype[0] = out_dtype;
    g.ct_begin[0] = 0;
    g.ct_begin[1] = N / TILE_N;
    g.n = 1;
    return launch_gemm_large_grouped(g, xq, x_scale, M, K, s);
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
