// gemm_lprog.cu -- LARGE programs: a list of stages with M > 16 tokens, each Eq. 4 end to end,
// in ONE persistent tcgen05 launch (lprogram.h).  The per-stage work is gemm_large_kernel's (same tiles, same warp
// roles, same pipeline); what is new is that the launch does not end between stages:
//   * activation quant is FUSED: before a stage's tiles, the eight decode warps of every CTA quantise the rows
//     r = blockIdx.x, += gridDim.x of x into the stage's int8 matrix and its alpha vector (quant.cuh's exact fast
//     quantiser), then the CTA counts itself in qdone[s]; the X producer (TMA) and the epilogue warps start the stage when
//     qdone[s] == gridDim.x.  The packed weights of the stage are already streaming (they depend on nothing).
//   * a stage with depends = 1 reads what earlier stages wrote: its quantisation waits for gdone[s-1] == gridDim.x, which
//     every CTA counts after its epilogue warps have stored their last tile of stage s-1.
// Against one act_quant launch + one GEMM launch per stage this removes two launch gaps, two prologues and one drain per
// stage (measured: DESIGN.md 6c).  All CTAs wait for each other: the grid must be co-resident (checked at build time).
#include <cuda.h>
#include <cuda_bf16.h>
#include "common.cuh"
#include "quant.cuh"
#include "gemm_large.cuh"
#include "lprogram.h"

namespace vla {

constexpr int LP_QT = 256;                               // quantising threads: the eight decode warps
constexpr int LP_QV = 6;                                 // vectors of 8 bf16 a thread holds per round
constexpr int LP_QROWS = 16;                             // most rows per round
static_assert(LP_EXTRA_SMEM == LP_QROWS * 4 + LP_QROWS * 16, "lprogram.h");

__device__ __forceinline__ void lp_bar(int id, int threads) {
    asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(threads) : "memory");
}

// rows blockIdx.x, += gridDim.x of the stage's x -> int8 + alpha.  Flat tasks of one 8-element vector; a round covers as
// many rows as fit LP_QT * LP_QV vectors, the vectors stay in registers between the absmax and the quantisation.
__device__ __forceinline__ void lp_quant_stage(const LpStage& st, int tid, unsigned* s_rowmax, float4* s_scale) {
    const int grid = (int)gridDim.x, cta = (int)blockIdx.x, nvec = st.K >> 3;
    const int R = st.M > cta ? (st.M - cta + grid - 1) / grid : 0;
    const int G = min(LP_QROWS, (LP_QT * LP_QV) / nvec);
    uint2* __restrict__ xq = reinterpret_cast<uint2*>(st.xq);
    for (int i0 = 0; i0 < R; i0 += G) {
        const int g = min(G, R - i0), ntask = g * nvec;
        if (tid < LP_QROWS) s_rowmax[tid] = 0u;
        lp_bar(2, LP_QT);
        uint4 v[LP_QV];
        int rl[LP_QV];
        size_t at[LP_QV];
#pragma unroll
        for (int j = 0; j < LP_QV; ++j) {
            const int f = tid + j * LP_QT;
            rl[j] = -1;
            at[j] = 0;
            v[j] = make_uint4(0, 0, 0, 0);
            if (f < ntask) {
                rl[j] = (int)__umulhi((unsigned)f, st.inv_nvec);
                at[j] = (size_t)(cta + (i0 + rl[j]) * grid) * nvec + (f - rl[j] * nvec);
                v[j] = __ldcg(st.x + at[j]);             // L2: another SM may have written it earlier in this launch
            }
        }
#pragma unroll
        for (int j = 0; j < LP_QV; ++j) {
            uint32_t m = absmax8_packed(v[j], 0u);
            m = max(m & 0xFFFFu, m >> 16);
            const int r0 = __shfl_sync(0xFFFFFFFFu, rl[j], 0);
            if (__all_sync(0xFFFFFFFFu, rl[j] == r0)) {
                m = __reduce_max_sync(0xFFFFFFFFu, m);
                if ((tid & 31) == 0 && r0 >= 0) atomicMax(s_rowmax + r0, m);
            } else if (rl[j] >= 0) {
                atomicMax(s_rowmax + rl[j], m);
            }
        }
        lp_bar(2, LP_QT);
        if (tid < g) {
            const float alpha = alpha_of(bf16lo(s_rowmax[tid]));
            s_scale[tid] = quant_scales_of_alpha(alpha);
            st.xs[cta + (i0 + tid) * grid] = alpha;
        }
        lp_bar(2, LP_QT);
#pragma unroll
        for (int j = 0; j < LP_QV; ++j)
            if (rl[j] >= 0) xq[at[j]] = quant8_fast(v[j], s_scale[rl[j]]);
    }
}

template <int KS>
__global__ void __launch_bounds__(LG_THREADS, 1) lprog_kernel(const __grid_constant__ DevLProg P) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* base_ptr = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t x_tile = P.x_tile;
    const uint32_t stride = KS * (LG_A_BYTES + x_tile);               // [A x KS | X x KS]
    constexpr uint32_t X_OFF = KS * LG_A_BYTES;
    constexpr uint32_t W_STAGE = KS * LG_W_BYTES;
    const uint32_t ns = (uint32_t)P.NS;
    const uint32_t sS = base;
    const uint32_t sW = sS + ns * stride;
    const uint32_t sBar = sW + LG_SW * W_STAGE + LG_SCALE_BYTES;
    uint8_t* pS = base_ptr;
    uint8_t* pW = base_ptr + (size_t)ns * stride;
    float* pScale = reinterpret_cast<float*>(pW + LG_SW * W_STAGE);
    auto bar_full_w = [&](uint32_t s) { return sBar + 8u * s; };
    auto bar_empty_w = [&](uint32_t s) { return sBar + 8u * (LG_SW + s); };
    auto bar_full = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + s); };
    auto bar_empty = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + LG_NS_MAX + s); };
    auto bar_acc_full = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + 2 * LG_NS_MAX + s); };
    auto bar_acc_empty = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + 2 * LG_NS_MAX + 2 + s); };
    const uint32_t tmem_slot = sBar + 8u * LG_NBAR;
    uint8_t* p_tail = base_ptr + (tmem_slot - base);
    volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(p_tail);
    unsigned* s_rowmax = reinterpret_cast<unsigned*>(p_tail + 16);
    float4* s_scale = reinterpret_cast<float4*>(p_tail + 16 + LP_QROWS * 4);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned grid = gridDim.x;
    const LpStage* __restrict__ stages = P.stages;

    if (threadIdx.x == 0) {
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
    pdl_launch_dependents();

    if (warp == 0) {
        // ---------------- W producer: runs ahead across stage boundaries (weights depend on nothing) ----------------
        if (lane < 4 * KS) {
            const int piece = lane & 3, kk = lane >> 2;
            uint32_t it = 0;
            for (int sidx = 0; sidx < P.n_stages; ++sidx) {
                const LpStage& st = stages[sidx];
                const int num_kb = st.K / TILE_K, tiles_n = st.tiles_n, ntiles = st.ntiles, nlin = st.grp.n;
                for (int tile = blockIdx.x; tile < ntiles; tile += grid) {
                    const int ct = tile % tiles_n;
                    int li = 0;
                    for (int j = 1; j < nlin; ++j) if (ct >= st.grp.ct_begin[j]) li = j;
                    const int nb = ct - st.grp.ct_begin[li];
                    const uint8_t* wsrc = st.grp.packed[li] + (size_t)(nb * 4 + piece) * num_kb * 1024;
                    for (int kb = 0; kb < num_kb; kb += KS, ++it) {
                        const uint32_t s = it % LG_SW;
                        if (it >= LG_SW) mbar_wait(bar_empty_w(s), ((it / LG_SW) & 1) ^ 1);
                        if (lane == 0) mbar_arrive_expect_tx(bar_full_w(s), W_STAGE);
                        __syncwarp((1u << (4 * KS)) - 1u);
                        tma_bulk_g2s(sW + s * W_STAGE + kk * LG_W_BYTES + piece * 1024, wsrc + (size_t)(kb + kk) * 1024, 1024, bar_full_w(s));
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ---------------- X producer: a stage's activations exist once every CTA has quantised its rows ----------------
        if (lane == 0) {
            uint32_t it = 0;
            bool waited = false;
            for (int sidx = 0; sidx < P.n_stages; ++sidx) {
                const LpStage& st = stages[sidx];
                const int num_kb = st.K / TILE_K, tiles_n = st.tiles_n, ntiles = st.ntiles, TN = st.TN;
                if ((int)blockIdx.x >= ntiles) continue;
                tma_prefetch_desc(st.tmap);
                if (!waited) { pdl_wait(); waited = true; }   // the counters are re-zeroed by the previous run's last CTA
                spin_until(P.qdone + sidx, grid);
                asm volatile("fence.proxy.async.global;" ::: "memory");       // generic-proxy stores -> TMA reads
                for (int tile = blockIdx.x; tile < ntiles; tile += grid) {
                    const int m0 = (tile / tiles_n) * TN;
                    for (int kb = 0; kb < num_kb; kb += KS, ++it) {
                        const uint32_t s = it % ns;
                        if (it >= ns) mbar_wait(bar_empty(s), ((it / ns) & 1) ^ 1);
                        mbar_arrive_expect_tx(bar_full(s), (uint32_t)KS * TN * TILE_K);
#pragma unroll
                        for (int kk = 0; kk < KS; ++kk)
                            tma_tensor2d_g2s(sS + s * stride + X_OFF + kk * x_tile, st.tmap, (kb + kk) * TILE_K, m0, bar_full(s));
                    }
                }
            }
        }
    } else if (warp == 2) {
        // ---------------- MMA issuer ----------------
        if (lane == 0) {
            uint32_t it = 0, ti = 0;
            for (int sidx = 0; sidx < P.n_stages; ++sidx) {
                const LpStage& st = stages[sidx];
                const int num_kb = st.K / TILE_K, ntiles = st.ntiles;
                const uint32_t idesc = umma_idesc_i8(TILE_N, st.TN);
                for (int tile = blockIdx.x; tile < ntiles; tile += grid, ++ti) {
                    const uint32_t ab = ti & 1;
                    if (ti >= 2) mbar_wait(bar_acc_empty(ab), ((ti >> 1) & 1) ^ 1);
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_base + ab * 256u;
                    for (int kb = 0; kb < num_kb; kb += KS, ++it) {
                        const uint32_t s = it % ns;
                        mbar_wait(bar_full(s), (it / ns) & 1);
                        tc_fence_after();
#pragma unroll
                        for (int kk = 0; kk < KS; ++kk) {
                            const uint64_t a_desc = umma_desc_k_sw128(sS + s * stride + kk * LG_A_BYTES);
                            const uint64_t b_desc = umma_desc_k_sw128(sS + s * stride + X_OFF + kk * x_tile);
#pragma unroll
                            for (int k = 0; k < TILE_K / 32; ++k)
                                mma_i8_ss(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | kk | k) != 0);
                        }
                        mma_commit(bar_empty(s));
                    }
                    mma_commit(bar_acc_full(ab));
                }
            }
        }
    } else if (warp <= 10) {
        // ---------------- decode warps: fused quant of the stage, then the stage's weight tiles ----------------
        const int dgrp = (warp - 3) >> 2;
        const int d = (threadIdx.x - 96) & 127, qt = (int)threadIdx.x - 96;
        const int t = d & 3, p = (d >> 2) & 1, q = (d >> 3) & 3, i32 = d >> 5;
        const int g = 2 * q + p;
        uint32_t it = 0;
        pdl_wait();                                           // x of the first stages may be the previous kernel's output
        for (int sidx = 0; sidx < P.n_stages; ++sidx) {
            const LpStage& st = stages[sidx];
            if (qt == 0 && st.wait_stage >= 0) spin_until(P.gdone + st.wait_stage, grid);
            lp_bar(2, LP_QT);
            lp_quant_stage(st, qt, s_rowmax, s_scale);
            lp_bar(2, LP_QT);                                 // every row of this CTA is stored ...
            if (qt == 0) red_release_gpu(P.qdone + sidx, 1u); // ... and published
            const int num_kb = st.K / TILE_K, ntiles = st.ntiles;
            for (int tile = blockIdx.x; tile < ntiles; tile += grid) {
                for (int kb = 0; kb < num_kb; kb += KS, ++it) {
                    if ((int)(it & 1u) != dgrp) continue;
                    const uint32_t sw = it % LG_SW, s = it % ns;
                    mbar_wait(bar_full_w(sw), (it / LG_SW) & 1);
                    const uint8_t* wst = pW + sw * W_STAGE;
                    uint4 wv[KS][2];
#pragma unroll
                    for (int kk = 0; kk < KS; ++kk)
#pragma unroll
                        for (int itx = 0; itx < 2; ++itx)
                            wv[kk][itx] = *reinterpret_cast<const uint4*>(wst + kk * LG_W_BYTES + ((i32 * 2 + (p ^ itx)) * 32 + g * 4 + t) * 16);
                    if (it >= ns) mbar_wait(bar_empty(s), ((it / ns) & 1) ^ 1);
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
                    fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) {
                        mbar_arrive(bar_empty_w(sw));
                        mbar_arrive(bar_full(s));
                    }
                }
            }
        }
    } else {
        // ---------------- epilogue warps ----------------
        const int lq = warp & 3;
        float* sc = pScale + lq * 256;
        const uint32_t sc_addr = sW + LG_SW * W_STAGE + (uint32_t)lq * 1024u;
        pdl_wait();                                           // the outputs may still be read by the previous kernel
        uint32_t ti = 0;
        for (int sidx = 0; sidx < P.n_stages; ++sidx) {
            const LpStage& st = stages[sidx];
            const int tiles_n = st.tiles_n, ntiles = st.ntiles, TN = st.TN, M = st.M, nlin = st.grp.n;
            if ((int)blockIdx.x < ntiles) {
                if (lane == 0) spin_until(P.qdone + sidx, grid);              // alpha of every row is stored
                __syncwarp();
            }
            const float* __restrict__ x_scale = st.xs;
            for (int tile = blockIdx.x; tile < ntiles; tile += grid, ++ti) {
                const int ct = tile % tiles_n, m0 = (tile / tiles_n) * TN;
                int li = 0;
                for (int j = 1; j < nlin; ++j) if (ct >= st.grp.ct_begin[j]) li = j;
                const int nb = ct - st.grp.ct_begin[li], N = st.grp.N[li], out_dtype = st.grp.dtype[li];
                void* __restrict__ out = st.grp.out[li];
                const float beta = (out_dtype == 2) ? 0.0f : __ldcg(st.grp.beta[li]);
                const uint32_t ab = ti & 1;
                const int ch = nb * TILE_N + lq * 32 + lane;
                if (out_dtype != 2)
                    for (int i = lane; i < TN; i += 32) sc[i] = (m0 + i < M) ? __fmul_rn(__ldcg(x_scale + m0 + i), beta) : 0.0f;
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
                    float sv[16];
#pragma unroll
                    for (int i4 = 0; i4 < 4; ++i4) {
                        const uint4 q4 = lds128_nv(sc_addr + (uint32_t)(c0 + 4 * i4) * 4u);
                        sv[4 * i4] = __uint_as_float(q4.x); sv[4 * i4 + 1] = __uint_as_float(q4.y);
                        sv[4 * i4 + 2] = __uint_as_float(q4.z); sv[4 * i4 + 3] = __uint_as_float(q4.w);
                    }
                    int acc[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) acc[i] = (int)r[i] >> 6;
                    const size_t o0 = (size_t)(m0 + c0) * N + ch;
                    if (nrow == 16) {
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
                    } else {
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
                if (lane == 0) mbar_arrive(bar_acc_empty(ab));
            }
            lp_bar(3, 128);                                   // the four epilogue warps have stored the CTA's tiles of the stage
            if (threadIdx.x == 11 * 32) red_release_gpu(P.gdone + sidx, 1u);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc(tmem_base, 512u);
    // the last CTA past its final counter access re-zeroes the counters for the next run of this program
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(P.done, 1u) == grid - 1u) {
            for (int s = 0; s < P.n_stages; ++s) { P.qdone[s] = 0u; P.gdone[s] = 0u; }
            *P.done = 0u;
            __threadfence();
        }
    }
}

cudaError_t lprogram_max_ctas_per_sm(int KS, int smem_bytes, int* out) {
    cudaError_t e;
    if (KS == 2) {
        e = cudaFuncSetAttribute(lprog_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
        if (e != cudaSuccess) return e;
        return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, lprog_kernel<2>, LG_THREADS, (size_t)smem_bytes);
    }
    e = cudaFuncSetAttribute(lprog_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, lprog_kernel<1>, LG_THREADS, (size_t)smem_bytes);
}

cudaError_t launch_lprogram(const DevLProg& prog, int grid, cudaStream_t s) {
    cudaError_t e = prog.KS == 2
        ? cudaFuncSetAttribute(lprog_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, prog.smem_bytes)
        : cudaFuncSetAttribute(lprog_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, prog.smem_bytes);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(LG_THREADS);
    cfg.dynamicSmemBytes = (size_t)prog.smem_bytes;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    count_launch();
    if (prog.KS == 2) return cudaLaunchKernelEx(&cfg, lprog_kernel<2>, prog);
    return cudaLaunchKernelEx(&cfg, lprog_kernel<1>, prog);
}

}  // namespace vla
