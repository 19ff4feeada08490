// gemm_lprog.cu -- LARGE programs: a list of stages with M > 16 tokens, each Eq. 4 end to end,
// in ONE persistent tcgen05 launch (lprogram.h).  The per-stage work is gemm_large_kernel's (same tiles, same warp
// roles, same pipeline); what is new is that the launch does not end between stages:
//   * activation quant is FUSED: dedicated quantiser warps of every CTA (after gemm_large_kernel's 15) quantise the rows
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

#ifndef VLA_LP_QG
#define VLA_LP_QG 1
#endif
#ifndef VLA_LP_QW
#define VLA_LP_QW 8
#endif
constexpr int LP_QG = VLA_LP_QG;                         // quantiser groups (after the 15 warps of gemm_large_kernel): group i
                                                         // takes the stages s = i (mod LP_QG), so LP_QG latency chains overlap
constexpr int LP_QW = VLA_LP_QW;                         // warps per group
constexpr int LP_QT = 32 * LP_QW;
constexpr int LP_THREADS = LG_THREADS + LP_QG * LP_QT + 32;         // + the publisher warp
constexpr int LP_QROWS = 16;                             // most rows per round
constexpr int LP_NBAR = LG_NBAR + 2 * LP_NA_MAX;          // + the A ring of the ATM form (full / empty)
static_assert(LP_QG == 1 && LP_EXTRA_SMEM >= LP_QROWS * 4 + LP_QROWS * 16 + 16 + 128, "lprogram.h");

#ifdef VLA_LP_STAMPS
__device__ __forceinline__ unsigned long long lp_now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
#define LP_STAMP(k) do { P.stamps[((size_t)sidx * gridDim.x + blockIdx.x) * 8 + (k)] = lp_now(); } while (0)
#else
#define LP_STAMP(k) do { } while (0)
#endif

// Tile t of a stage runs on CTA (t + rot) mod grid.  The host picks `rot` per stage from its per-CTA load table (api_program.cu):
// the stage's first wave starts on the least-loaded window of CTAs, so the CTAs a short stage leaves idle are the first to
// start the next one (independent stages overlap) and long tiles do not queue up behind each other.
__device__ __forceinline__ int lp_first_tile(const LpStage& st, unsigned grid) {
    const int b = (int)blockIdx.x, r = st.rot;
    return b >= r ? b - r : b + (int)grid - r;
}
__device__ __forceinline__ void lp_bar(int id, int threads) {
    asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(threads) : "memory");
}

// rows blockIdx.x, += gridDim.x of the stage's x -> int8 + alpha.  The rows are STAGED IN SHARED MEMORY: one bulk copy (TMA)
// per row, all rows of a chunk in flight at once, then the absmax pass and the quantising pass both read shared memory.  x is
// read from L2 / DRAM exactly once, no registers are held across the passes, and the memory parallelism does not depend on
// how many 16-byte loads a thread can keep in flight (the register-held form took 10-11 us per stage at K = 6912).
// The row buffer is DOUBLE-BUFFERED whenever a row fits half of it: while the threads work on chunk c (half c & 1), thread 0
// already has the copies of chunk c + 1 in flight into the other half -- the next rows of the same stage, or the FIRST rows of
// the next stage if that stage's inputs are already cleared (s_gok).  In steady state the quantiser is the pacing chain of a
// large program (its stages follow each other without a gap), and the 1-1.5 us a stage used to wait for its rows were a
// fifth of that chain.
struct LpQuantArgs {           // the quantiser's view of a stage, read from the table BEFORE it waits for the stage's inputs
    const uint4* x;
    uint2* xq;
    float* xs;
    int nvec, wait_stage, R, rpc;       // R = rows of this CTA, rpc = rows per chunk
    bool dbl, x_dep;
};
__device__ __forceinline__ LpQuantArgs lp_quant_args(const LpStage& st) {
    LpQuantArgs a;
    a.x = st.x; a.xq = reinterpret_cast<uint2*>(st.xq); a.xs = st.xs;
    a.nvec = st.K >> 3; a.wait_stage = st.wait_stage;
    a.R = st.q_rows + ((int)blockIdx.x < st.q_rem ? 1 : 0); a.rpc = st.q_rpc; a.dbl = st.q_dbl != 0; a.x_dep = st.x_dep != 0;
    return a;
}
// lane 0 of quantiser warp w: the bulk copies of rows i0 + w, i0 + w + 8, ... (< i0 + g, of this CTA's rows) of a stage -> the
// row buffer at `dst`; warp 0 also announces the bytes.  (One thread issuing all copies of a chunk kept the other 255 waiting
// for ~70 cycles per copy.)
__device__ __forceinline__ void lp_quant_issue(const LpQuantArgs& a, int i0, int g, uint32_t dst, uint32_t bar, int warp) {
    const int grid = (int)gridDim.x, cta = (int)blockIdx.x;
    const uint32_t row_bytes = (uint32_t)a.nvec * 16u;
    if (a.x_dep) asm volatile("fence.proxy.async.global;" ::: "memory");      // x written by other SMs -> this thread's bulk copies
    if (warp == 0) mbar_arrive_expect_tx(bar, (uint32_t)g * row_bytes);
    for (int j = warp; j < g; j += LP_QW)
        tma_bulk_g2s(dst + (uint32_t)j * row_bytes, a.x + (size_t)(cta + (i0 + j) * grid) * a.nvec, row_bytes, bar);
}

// c = chunks this CTA has processed so far (all stages); inflight = the copies of chunk c are already issued (a prefetch)
__device__ __forceinline__ void lp_quant_stage(const LpQuantArgs& a, const LpQuantArgs* nx, int sidx, uint32_t s_gok, uint32_t s_pf,
                                               int tid, int bar_id, unsigned* s_rowmax, float4* s_scale, uint32_t qbuf,
                                               uint32_t qbuf_bytes, uint32_t bar_q, uint32_t& c, bool& inflight, unsigned long long* dbg) {
    const int grid = (int)gridDim.x, cta = (int)blockIdx.x, nvec = a.nvec, warp = tid >> 5, lane = tid & 31;
    const uint32_t row_bytes = (uint32_t)nvec * 16u, half = (qbuf_bytes >> 1) & ~127u;
    uint2* __restrict__ xq = a.xq;
    float* __restrict__ xs = a.xs;
    for (int i0 = 0; i0 < a.R; i0 += a.rpc, ++c) {
        const int g = min(a.rpc, a.R - i0);
        const uint32_t buf = qbuf + ((a.dbl && (c & 1u)) ? half : 0u), bar = bar_q + 8u * (c & 1u);
        if (tid == 0) {
            if (i0 == 0 && a.wait_stage >= 0 && !inflight) {          // cleared by the publisher warp, usually during the last stage
                const long long t0 = clock64();
                unsigned ok;
                do {
                    asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(ok) : "r"(s_gok) : "memory");
                    if (clock64() - t0 > (1ll << 32)) __trap();
                } while (ok <= (unsigned)sidx);
            }
            // what to load DURING this chunk, into the other half (read last by chunk c - 1): 1 = the next chunk of this stage,
            // 2 = the first chunk of the next stage, if that stage is already cleared (never waits)
            unsigned pf = 0u;
            if (a.dbl) {
                if (i0 + a.rpc < a.R) pf = 1u;
                else if (nx != nullptr && nx->dbl && nx->R > 0) {
                    bool ok = nx->wait_stage < 0;
                    if (!ok) {
                        unsigned have;
                        asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(have) : "r"(s_gok) : "memory");
                        ok = have > (unsigned)(sidx + 1);
                    }
                    if (ok) pf = 2u;
                }
            }
            asm volatile("st.shared::cta.u32 [%0], %1;" :: "r"(s_pf), "r"(pf) : "memory");
        }
        if (tid < LP_QROWS) s_rowmax[tid] = 0u;
        lp_bar(bar_id, LP_QT);                                        // (also: everybody is done reading the previous chunk)
        unsigned pf;
        asm volatile("ld.shared::cta.u32 %0, [%1];" : "=r"(pf) : "r"(s_pf) : "memory");
        if (lane == 0) {
            if (!inflight) lp_quant_issue(a, i0, g, buf, bar, warp);
            if (pf != 0u) {
                const uint32_t nbuf = qbuf + ((c & 1u) ? 0u : half), nbar = bar_q + 8u * ((c + 1u) & 1u);
                if (pf == 1u) lp_quant_issue(a, i0 + a.rpc, min(a.rpc, a.R - i0 - a.rpc), nbuf, nbar, warp);
                else lp_quant_issue(*nx, 0, min(nx->rpc, nx->R), nbuf, nbar, warp);
            }
        }
        inflight = pf != 0u;
        mbar_wait(bar, (c >> 1) & 1u);
#ifdef VLA_LP_STAMPS
        if (tid == 0 && i0 == 0) dbg[6] = lp_now();
#endif
        // Row r of the chunk belongs to the tpr = LP_QT / rp consecutive threads r * tpr .. (rp = g rounded up to a power of
        // two: 256 .. 16 threads per row), thread j of them takes vectors j, j + tpr, ...: a thread stays in ONE row, so
        // the loops carry no warp collectives, no index division and no per-vector scale lookup.
        const int lg = 32 - __clz(g - 1);                             // rp = 2^lg >= g (g <= 16)
        static_assert(LP_QT == 256, "shifts below");
        const int tpr = LP_QT >> lg, my_row = tid >> (8 - lg), j = tid & (tpr - 1);
        const bool mine = my_row < g;
        const uint32_t row_s = buf + (uint32_t)my_row * row_bytes;
        uint32_t m = 0u;
        if (mine) {
#pragma unroll 4
            for (int v = j; v < nvec; v += tpr) m = absmax8_packed(lds128_nv(row_s + (uint32_t)v * 16u), m);   // pass 1
        }
        m = max(m & 0xFFFFu, m >> 16);
        if (tpr >= 32) {
            m = __reduce_max_sync(0xFFFFFFFFu, m);
            if ((tid & 31) == 0 && mine) atomicMax(s_rowmax + my_row, m);
        } else {                                                      // 16 threads per row: two rows per warp
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
            if ((tid & 15) == 0 && mine) atomicMax(s_rowmax + my_row, m);
        }
        lp_bar(bar_id, LP_QT);
#ifdef VLA_LP_STAMPS
        if (tid == 0 && i0 == 0) dbg[7] = lp_now();
#endif
        if (tid < g) {
            const float alpha = alpha_of(bf16lo(s_rowmax[tid]));
            s_scale[tid] = quant_scales_of_alpha(alpha);
            xs[cta + (i0 + tid) * grid] = alpha;
        }
        lp_bar(bar_id, LP_QT);
        if (mine) {
            const float4 sc = s_scale[my_row];
            uint2* __restrict__ dst = xq + (size_t)(cta + (i0 + my_row) * grid) * nvec;
#pragma unroll 2
            for (int v = j; v < nvec; v += tpr) dst[v] = quant8_fast(lds128_nv(row_s + (uint32_t)v * 16u), sc);      // pass 2
        }
    }
}

template <int KS, bool ATM>
__global__ void __launch_bounds__(LP_THREADS, 1) lprog_kernel(const __grid_constant__ DevLProg P) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* base_ptr = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t x_tile = P.x_tile;
    // ATM: the decoded A operand lives in TENSOR MEMORY (columns behind the two accumulators, NA stages of KS x 32 columns),
    // and a shared-memory pipeline stage holds X only -- so many more X tiles are in flight for the same shared memory
    const uint32_t stride = KS * ((ATM ? 0u : (uint32_t)LG_A_BYTES) + x_tile);   // [A x KS | X x KS], ATM: [X x KS]
    constexpr uint32_t X_OFF = ATM ? 0u : KS * LG_A_BYTES;
    const uint32_t acc_stride = ATM ? (uint32_t)P.acc_stride : 256u;  // TMEM columns between the two accumulators
    const uint32_t a_col0 = 2u * acc_stride;                          // ATM: first column of the A ring
    const uint32_t na = (uint32_t)P.NA;
    constexpr uint32_t W_STAGE = KS * LG_W_BYTES;
    const uint32_t ns = (uint32_t)P.NS;
    const uint32_t sS = base;
    const uint32_t sW = sS + ns * stride;
    const uint32_t nsw = (uint32_t)P.NSW;                               // packed-weight stages in use (<= LG_SW)
    const uint32_t sBar = sW + nsw * W_STAGE + LG_SCALE_BYTES;
    uint8_t* pS = base_ptr;
    uint8_t* pW = base_ptr + (size_t)ns * stride;
    float* pScale = reinterpret_cast<float*>(pW + nsw * W_STAGE);
    auto bar_full_w = [&](uint32_t s) { return sBar + 8u * s; };
    auto bar_empty_w = [&](uint32_t s) { return sBar + 8u * (LG_SW + s); };
    auto bar_full = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + s); };
    auto bar_empty = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + LG_NS_MAX + s); };
    auto bar_acc_full = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + 2 * LG_NS_MAX + s); };
    auto bar_acc_empty = [&](uint32_t s) { return sBar + 8u * (2 * LG_SW + 2 * LG_NS_MAX + 2 + s); };
    auto bar_afull = [&](uint32_t s) { return sBar + 8u * (LG_NBAR + s); };                   // ATM: A stage written to TMEM
    auto bar_aempty = [&](uint32_t s) { return sBar + 8u * (LG_NBAR + LP_NA_MAX + s); };      // ATM: its MMAs are done
    const uint32_t tmem_slot = sBar + 8u * LP_NBAR;
    uint8_t* p_tail = base_ptr + (tmem_slot - base);
    volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(p_tail);
    unsigned* s_rowmax = reinterpret_cast<unsigned*>(p_tail + 16);
    float4* s_scale = reinterpret_cast<float4*>(p_tail + 16 + LP_QROWS * 4);
    const uint32_t s_qcount = tmem_slot + 8u;                // quantiser warps that have stored a stage, summed over the stages
    const uint32_t s_gok = tmem_slot + 12u;                  // stages the publisher has cleared for the quantiser
    const uint32_t s_pf = tmem_slot + 4u;                    // the quantiser's prefetch decision of the current chunk
    const uint32_t bar_q = tmem_slot + 16u + LP_QROWS * 20u;  // the quantiser's row copies have landed
    const uint32_t qbuf = (bar_q + 16u + 127u) & ~127u;       // row buffer of the quantiser, P.qbuf_bytes

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned grid = gridDim.x;
    const LpStage* __restrict__ stages = P.stages;

    if (threadIdx.x == 0) {
        for (int s = 0; s < LG_SW; ++s) { mbar_init(bar_full_w(s), 1); mbar_init(bar_empty_w(s), 4); }
        for (int s = 0; s < LG_NS_MAX; ++s) { mbar_init(bar_full(s), ATM ? 1 : 5); mbar_init(bar_empty(s), 1); }
        for (int s = 0; s < LP_NA_MAX; ++s) { mbar_init(bar_afull(s), 4); mbar_init(bar_aempty(s), 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(bar_acc_full(s), 1); mbar_init(bar_acc_empty(s), 4); }
        mbar_init(sBar + 8u * LP_NBAR + 16u + LP_QROWS * 20u, 1);         // bar_q: one per half of the quantiser's row buffer
        mbar_init(sBar + 8u * LP_NBAR + 16u + LP_QROWS * 20u + 8u, 1);
        fence_barrier_init();
        asm volatile("st.shared::cta.u32 [%0], %1;" :: "r"(tmem_slot + 8u), "r"(0u) : "memory");
        asm volatile("st.shared::cta.u32 [%0], %1;" :: "r"(tmem_slot + 12u), "r"(0u) : "memory");
    }
    if (warp == 2) tmem_alloc(tmem_slot, 512u);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_launch_dependents();

    if (warp == 0) {
        // ---------------- W producer: runs ahead across stage boundaries (weights depend on nothing) ----------------
        if (lane < 4) {                                       // one copy per 32-channel piece: its KS k blocks are contiguous
            const int piece = lane;
            uint32_t it = 0;
            RingCur cw;
            for (int sidx = 0; sidx < P.n_stages; ++sidx) {
                const LpStage& st = stages[sidx];
                const int num_kb = st.K / TILE_K, tiles_n = st.tiles_n, ntiles = st.ntiles, nlin = st.grp.n;
                for (int tile = lp_first_tile(st, grid); tile < ntiles; tile += grid) {
                    const int ct = tile % tiles_n;
                    int li = 0;
                    for (int j = 1; j < nlin; ++j) if (ct >= st.grp.ct_begin[j]) li = j;
                    const int nb = ct - st.grp.ct_begin[li];
                    const uint8_t* wsrc = st.grp.packed[li] + (size_t)(nb * 4 + piece) * num_kb * 1024;
                    for (int kb = 0; kb < num_kb; kb += KS, ++it, cw.next(nsw)) {
                        const uint32_t s = cw.s;
                        if (cw.wrapped) mbar_wait(bar_empty_w(s), cw.ph ^ 1u);
                        if (lane == 0) mbar_arrive_expect_tx(bar_full_w(s), W_STAGE);
                        __syncwarp(0xFu);
                        tma_bulk_g2s(sW + s * W_STAGE + piece * (KS * 1024), wsrc + (size_t)kb * 1024, KS * 1024, bar_full_w(s));
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ---------------- X producer: a stage's activations exist once every CTA has quantised its rows ----------------
        if (lane == 0) {
            uint32_t it = 0;
            RingCur cx;
            bool waited = false;
            for (int sidx = 0; sidx < P.n_stages; ++sidx) {
                const LpStage& st = stages[sidx];
                const int num_kb = st.K / TILE_K, tiles_n = st.tiles_n, ntiles = st.ntiles, TN = st.TN;
                if (lp_first_tile(st, grid) >= ntiles) continue;
                tma_prefetch_desc(st.tmap);
                if (!waited) { pdl_wait(); waited = true; }   // the counters are re-zeroed by the previous run's last CTA
                spin_until(P.qdone + sidx, grid);
                LP_STAMP(2);
                asm volatile("fence.proxy.async.global;" ::: "memory");       // generic-proxy stores -> TMA reads
                for (int tile = lp_first_tile(st, grid); tile < ntiles; tile += grid) {
                    const int m0 = (tile / tiles_n) * TN;
                    for (int kb = 0; kb < num_kb; kb += KS, ++it, cx.next(ns)) {
                        const uint32_t s = cx.s;
                        if (cx.wrapped) mbar_wait(bar_empty(s), cx.ph ^ 1u);
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
            const uint64_t desc0 = umma_desc_k_sw128(sS);
            uint32_t it = 0, ti = 0;
            RingCur cm, ca;
            for (int sidx = 0; sidx < P.n_stages; ++sidx) {
                const LpStage& st = stages[sidx];
                const int num_kb = st.K / TILE_K, ntiles = st.ntiles;
                const uint32_t idesc = umma_idesc_i8(TILE_N, st.TN);
                for (int tile = lp_first_tile(st, grid); tile < ntiles; tile += grid, ++ti) {
                    const uint32_t ab = ti & 1;
                    if (ti >= 2) mbar_wait(bar_acc_empty(ab), ((ti >> 1) & 1) ^ 1);
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_base + ab * acc_stride;
                    for (int kb = 0; kb < num_kb; kb += KS, ++it, cm.next(ns), ca.next(na)) {
                        const uint32_t s = cm.s;
                        mbar_wait(bar_full(s), cm.ph);
                        if constexpr (ATM) mbar_wait(bar_afull(ca.s), ca.ph);
                        tc_fence_after();
                        if (kb == 0 && tile == lp_first_tile(st, grid)) LP_STAMP(3);
#pragma unroll
                        for (int kk = 0; kk < KS; ++kk) {
                            // (descriptor = constant fields + (shared address >> 4): only the address part moves)
                            const uint64_t b_desc = desc0 + ((s * stride + X_OFF + kk * x_tile) >> 4);
                            if constexpr (ATM) {
                                const uint32_t a_tmem = tmem_base + a_col0 + (ca.s * KS + kk) * 32u;
#pragma unroll
                                for (int k = 0; k < TILE_K / 32; ++k)
                                    mma_i8_ts(d_tmem, a_tmem + 8 * k, b_desc + 2 * k, idesc, (kb | kk | k) != 0);
                            } else {
                                const uint64_t a_desc = desc0 + ((s * stride + kk * LG_A_BYTES) >> 4);
#pragma unroll
                                for (int k = 0; k < TILE_K / 32; ++k)
                                    mma_i8_ss(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | kk | k) != 0);
                            }
                        }
                        if constexpr (ATM) mma_commit(bar_aempty(ca.s));
                        mma_commit(bar_empty(s));
                    }
                    mma_commit(bar_acc_full(ab));
                    LP_STAMP(4);
                }
            }
        }
    } else if (warp <= 10) {
        // ---------------- decode warps ----------------
        const int dgrp = (warp - 3) >> 2;
        const int d = (threadIdx.x - 96) & 127;
        const int t = d & 3, p = (d >> 2) & 1, q = (d >> 3) & 3, i32 = d >> 5;
        const int g = 2 * q + p;
        uint32_t it = 0;
            RingCur cd, cdw, cda;
        for (int sidx = 0; sidx < P.n_stages; ++sidx) {
            const LpStage& st = stages[sidx];
            const int num_kb = st.K / TILE_K, ntiles = st.ntiles;
            for (int tile = lp_first_tile(st, grid); tile < ntiles; tile += grid) {
                for (int kb = 0; kb < num_kb; kb += KS, ++it, cd.next(ns), cdw.next(nsw), cda.next(na)) {
                    if ((int)(it & 1u) != dgrp) continue;
                    const uint32_t sw = cdw.s, s = cd.s;
                    mbar_wait(bar_full_w(sw), cdw.ph);
                    const uint8_t* wst = pW + sw * W_STAGE;
                    if constexpr (ATM) {
                        // Thread l of the warp owns channel 32 * piece + l = TMEM lane (piece = warp & 3: the lane quarter this
                        // warp may access).  Its 128 k of a k block are the 8 words (h, t) of the piece, word (h, t) -> columns
                        // 16 h + 4 t .. + 3 (packed layout: common.cuh).
                        const int piece = warp & 3, jj = lane >> 3, gg = lane & 7;
                        uint32_t wr[KS][8];
#pragma unroll
                        for (int kk = 0; kk < KS; ++kk)
#pragma unroll
                            for (int u = 0; u < 8; ++u)
                                wr[kk][u] = *reinterpret_cast<const uint32_t*>(wst + piece * (KS * 1024) + kk * 1024 + ((((u >> 2) * 32 + gg * 4 + (u & 3)) * 4 + jj) * 4));
                        if (cda.wrapped) mbar_wait(bar_aempty(cda.s), cda.ph ^ 1u);
                        tc_fence_after();
#pragma unroll
                        for (int kk = 0; kk < KS; ++kk) {
                            uint32_t r[32];
#pragma unroll
                            for (int u = 0; u < 8; ++u) {
                                r[4 * u + 0] = decode64<0>(wr[kk][u]); r[4 * u + 1] = decode64<1>(wr[kk][u]);
                                r[4 * u + 2] = decode64<2>(wr[kk][u]); r[4 * u + 3] = decode64<3>(wr[kk][u]);
                            }
                            tmem_st_32x32b_x32(tmem_base + a_col0 + (cda.s * KS + kk) * 32u + ((uint32_t)(piece * 32) << 16), r);
                        }
                        tmem_st_wait();
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) {
                            mbar_arrive(bar_empty_w(sw));
                            mbar_arrive(bar_afull(cda.s));
                        }
                        continue;
                    }
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
                    fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) {
                        mbar_arrive(bar_empty_w(sw));
                        mbar_arrive(bar_full(s));
                    }
                }
            }
        }
    } else if (warp <= 14) {
        // ---------------- epilogue warps ----------------
        const int lq = warp & 3;
        float* sc = pScale + lq * 256;
        const uint32_t sc_addr = sW + nsw * W_STAGE + (uint32_t)lq * 1024u;
        pdl_wait();                                           // the outputs may still be read by the previous kernel
        uint32_t ti = 0;
        for (int sidx = 0; sidx < P.n_stages; ++sidx) {
            const LpStage& st = stages[sidx];
            const int tiles_n = st.tiles_n, ntiles = st.ntiles, TN = st.TN, M = st.M, nlin = st.grp.n;
            if (lp_first_tile(st, grid) < ntiles) {
                if (threadIdx.x == 11 * 32) spin_until(P.qdone + sidx, grid); // alpha of every row is stored
                lp_bar(3, 128);
            }
            const float* __restrict__ x_scale = st.xs;
            for (int tile = lp_first_tile(st, grid); tile < ntiles; tile += grid, ++ti) {
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
                const uint32_t t_addr = tmem_base + ab * acc_stride + ((uint32_t)(lq * 32) << 16);
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
            if (threadIdx.x == 11 * 32) { LP_STAMP(5); red_release_gpu(P.gdone + sidx, 1u); }
        }
    }
    else if (warp < 15 + LP_QW) {
        // ---------------- quantiser warps: run ahead of the GEMM as far as the stages' dependencies allow ----------------
        const int qt = (int)threadIdx.x - LG_THREADS;
        const int bar_id = 4;
        pdl_wait();                                           // x of the first stages may be the previous kernel's output
        LpQuantArgs next = lp_quant_args(stages[0]);
        LpQuantArgs next2 = lp_quant_args(stages[P.n_stages > 1 ? 1 : 0]);
        uint32_t q_chunk = 0u;
        bool q_inflight = false;
        for (int sidx = 0; sidx < P.n_stages; ++sidx) {
            const LpQuantArgs st = next;
            const bool has_next = sidx + 1 < P.n_stages;
            next = next2;
            if (sidx + 2 < P.n_stages) next2 = lp_quant_args(stages[sidx + 2]);      // two stages ahead: an L2 round trip off the chain
            if (qt == 0) LP_STAMP(0);
#ifdef VLA_LP_STAMPS
            lp_quant_stage(st, has_next ? &next : nullptr, sidx, s_gok, s_pf, qt, bar_id, s_rowmax, s_scale, qbuf, P.qbuf_bytes, bar_q,
                           q_chunk, q_inflight, P.stamps + ((size_t)sidx * gridDim.x + blockIdx.x) * 8);
#else
            lp_quant_stage(st, has_next ? &next : nullptr, sidx, s_gok, s_pf, qt, bar_id, s_rowmax, s_scale, qbuf, P.qbuf_bytes, bar_q,
                           q_chunk, q_inflight, nullptr);
#endif
            // this warp's rows of the stage are stored: tell the publisher warp and go on with the next stage -- the
            // gpu-scope release (a fence that waits for the stores, ~1 us) is the publisher's, off this chain
            __syncwarp();
            if (lane == 0) asm volatile("red.release.cta.shared::cta.add.u32 [%0], 1;" :: "r"(s_qcount) : "memory");
        }
    } else {
        // ---------------- publisher: the quantiser's grid-scope hand-offs, off its chain ----------------
        // (1) counts the CTA in qdone[s] once all quantiser warps have stored stage s;  (2) clears stage s+1 for the
        // quantiser (s_gok = stages cleared) once gdone[wait_stage(s+1)] == grid, polled WHILE the quantiser works on stage s.
        // Neither blocks the other: a stage that waits for an older stage's GEMM (interleaved chains, depends = d) must not
        // hold back the publication of the stage in between.
        if (lane == 0) {
            pdl_wait();                                       // the counters are re-zeroed by the previous run's last CTA
            const int n = P.n_stages;
            int qs = 0, gs = 1;                               // next stage to publish / to clear (stage 0 waits for nothing)
            asm volatile("st.release.cta.shared::cta.u32 [%0], %1;" :: "r"(s_gok), "r"(1u) : "memory");
            int w_gs = gs < n ? stages[gs].wait_stage : -1;
            long long t0 = clock64();
            while (qs < n) {
                unsigned have;
                asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(have) : "r"(s_qcount) : "memory");
                if (have >= (unsigned)LP_QW * (unsigned)(qs + 1)) {
                    const int sidx = qs;
                    LP_STAMP(1);
                    red_release_gpu(P.qdone + sidx, 1u);      // cumulative: covers the quantiser warps' stores observed above
                    ++qs;
                    t0 = clock64();
                    continue;
                }
                if (gs < n && gs <= qs + 1) {                 // one try (an L2 round trip), then back to the cheap check
                    if (w_gs < 0 || ld_acquire_gpu(P.gdone + w_gs) >= grid) {
                        ++gs;
                        asm volatile("st.release.cta.shared::cta.u32 [%0], %1;" :: "r"(s_gok), "r"((unsigned)gs) : "memory");
                        w_gs = gs < n ? stages[gs].wait_stage : -1;
                        t0 = clock64();
                    }
                }
                if (clock64() - t0 > (1ll << 32)) __trap();
            }
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

template <int KS, bool ATM>
static cudaError_t lp_prepare(int smem_bytes, int* occ_out) {
    cudaError_t e = cudaFuncSetAttribute(lprog_kernel<KS, ATM>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    if (e != cudaSuccess || !occ_out) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_out, lprog_kernel<KS, ATM>, LP_THREADS, (size_t)smem_bytes);
}
static cudaError_t lp_prepare_any(int KS, int atm, int smem_bytes, int* occ_out) {
    if (atm) return KS == 2 ? lp_prepare<2, true>(smem_bytes, occ_out) : lp_prepare<1, true>(smem_bytes, occ_out);
    return KS == 2 ? lp_prepare<2, false>(smem_bytes, occ_out) : lp_prepare<1, false>(smem_bytes, occ_out);
}

cudaError_t lprogram_max_ctas_per_sm(int KS, int atm, int smem_bytes, int* out) { return lp_prepare_any(KS, atm, smem_bytes, out); }

cudaError_t launch_lprogram(const DevLProg& prog, int grid, cudaStream_t s) {
    cudaError_t e = lp_prepare_any(prog.KS, prog.ATM, prog.smem_bytes, nullptr);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(LP_THREADS);
    cfg.dynamicSmemBytes = (size_t)prog.smem_bytes;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    count_launch();
    if (prog.ATM) {
        if (prog.KS == 2) return cudaLaunchKernelEx(&cfg, lprog_kernel<2, true>, prog);
        return cudaLaunchKernelEx(&cfg, lprog_kernel<1, true>, prog);
    }
    if (prog.KS == 2) return cudaLaunchKernelEx(&cfg, lprog_kernel<2, false>, prog);
    return cudaLaunchKernelEx(&cfg, lprog_kernel<1, false>, prog);
}

}  // namespace vla
