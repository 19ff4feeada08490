// gemm_program.cu -- persistent "program" kernel for the small-M (M <= 16) regime: ONE launch runs a whole list
// of ternary linears (Eq. 4), independent or chained, e.g. the 30-layer stack of
// BASELINE.json configs[3].  PAPER.md line 56 removes dispatch overhead by persisting graphs; on B200 a launch
// costs ~5000 cycles, more than ten times the HBM time of a 1.6 MB weight tensor, so the whole program is one
// kernel and the only thing that ever waits is data.
//
// Grid: one CTA per SM, 16 warps.
//   warp 15 (producer)   streams this CTA's share of the packed weights of EVERY stage, in program order, through
//                        a ring of 30 KiB shared-memory slots with cp.async.bulk (TMA) + mbarriers.  It starts before
//                        griddepcontrol.wait (weights never depend on the previous kernel) and never waits on
//                        activations, so HBM stays busy across launch, stage and phase boundaries.
//   warps 0-14 (consumers) per stage:
//     1. activation quant, Eq. 4 lines 1-2, FUSED INTO THE KERNEL (quant_rows): a SMALL stage (<= 1440 sixteen-element
//        tasks, e.g. M = 8 x K = 2560) is quantised by every CTA of its group for itself, from the bf16 rows straight
//        into shared memory in mma.m16n8k32 B-fragment order -- no int8 round trip, no flag, nothing to wait for.  A
//        LARGER stage is quantised cooperatively: row r once, by CTA r mod c of the stage's group, into the stage's
//        scratch (already in fragment order), published with one release per CTA; every CTA of the group then pulls the
//        finished fragments with one bulk copy.  Either way the weight ring is never gated on activations.
//        The quantiser is an exact shortcut of the two true divisions (bracketed FMA, true-division patch for the rare
//        element whose bracket holds a rounding boundary): bit-identical to quant.cuh / the oracle.
//     2. GEMM: packed words from the ring are decoded in registers (2 ALU ops per 4 weights, common.cuh) into A
//        fragments, B fragments come from shared memory, int32 accumulation on the warp-level int8 MMA.  Either
//        three TEAMS of five warps work on three granules at once (each team's warps split the k blocks of its
//        granule), or -- when the CTA has fewer than three granules of the stage -- all 15 warps split one granule.
//        Partial sums meet in an int32 tile in shared memory (red.shared.add: exact in any order).
//     3. dequant epilogue  y = (float)acc * (alpha_m * beta), fp32 / bf16 RNE / raw int32.
// Work unit: a GRANULE = 32 output channels x all of K of one linear (one contiguous run of 8*K bytes).  The stages
// of one PHASE are independent, so they run CONCURRENTLY on disjoint CTA groups sized by the program compiler
// (api_program.cu); granule gi of a stage goes to CTA (gi mod group size) of its group.
// Counters in the program buffer (re-zeroed by the last CTA of every launch):
//   bp[p]  = CTAs that finished phase p      (a dependent phase's CTAs wait for bp[p-1] == gridDim.x before reading x)
//   cnt[s] = rows of cooperative stage s in its scratch   (the stage's group waits for cnt[s] == M_s before its bulk copy)
// Every sum is an exact integer sum and the quantiser reproduces the two true divisions of Eq. 4 bit for bit, so the
// result is bit-identical to the per-call kernels and to the oracle.
#include <cuda_bf16.h>
#include "common.cuh"
#include "kernels.h"
#include "program.h"
#include "quant.cuh"

namespace vla {

// 15 consumer warps + 1 producer = 16 warps = 4 per SM sub-partition -> 128 registers per thread.
constexpr int PG_CONSUMERS = PG_W * 32;          // 480 threads
constexpr int PG_THREADS = PG_CONSUMERS + 32;    // 512
constexpr uint32_t INFO_STAGE = 0xFFFFu;         // s_info[phase]: the stage this CTA runs in the phase + 1 (0: none)
constexpr uint32_t INFO_PUBLISH = 1u << 17;      // DevStage.flags bit 1
static_assert(PG_TEAMS * PG_TW == PG_W, "teams must cover the consumer warps");

#ifdef VLA_PROG_STAMPS
// debug builds only: stamp k of this CTA (globaltimer ns) into the program buffer, 32 slots per CTA
#define PG_STAMP(k) do { if (threadIdx.x == 0 && P.stamps) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); P.stamps[blockIdx.x * 32 + (k)] = t_; } } while (0)
#else
#define PG_STAMP(k) do { } while (0)
#endif

__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;" :: "n"(PG_CONSUMERS) : "memory"); }
__device__ __forceinline__ void team_bar(int team) {
    asm volatile("bar.sync %0, %1;" :: "r"(2 + team), "n"(PG_TW * 32) : "memory");
}

__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr) : "memory");
    return r;
}
__device__ __forceinline__ void sts128(uint32_t addr, uint4 v) {
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" :: "r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ int lds32(uint32_t addr) {
    int r;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(r) : "r"(addr));
    return r;
}
__device__ __forceinline__ void sts32(uint32_t addr, int v) {
    asm volatile("st.shared.s32 [%0], %1;" :: "r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void red_shared_add(uint32_t addr, int v) {
    asm volatile("red.shared.add.s32 [%0], %1;" :: "r"(addr), "r"(v) : "memory");
}
// publish: every store this CTA made before the preceding consumer_bar() becomes visible before the count does
// non-volatile form: the compiler may interleave it with the decode of the next block
__device__ __forceinline__ void mma_m16n8k32_s8_nv(int (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                                   uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// ---------------------------------------------------------------- ring bookkeeping
// Chunk number `seq` of this CTA (in producer order, over all its stages) lives in slot seq % nslot, in ring round
// seq / nslot.  An mbarrier only tells the PARITY of a phase, so a consumer may wait for round r of a slot only once
// round r-1 of that slot has landed; teams skip over each other's chunks and could otherwise be two rounds ahead of a
// slot.  s_got[slot] = seq + 1 of the newest chunk of the slot whose arrival a consumer has seen: the consumer of chunk
// seq first waits for s_got[slot] >= seq + 1 - nslot, then on the mbarrier.
struct Ring { uint32_t base, slot_bytes, nslot, bar_full, bar_empty, got; };
struct RingPos { uint32_t slot, parity; };
__device__ __forceinline__ RingPos ring_pos(uint32_t seq, uint32_t nslot) {
    const uint32_t round = seq / nslot;
    return RingPos{seq - round * nslot, round & 1u};
}
__device__ __forceinline__ RingPos ring_wait(const Ring& R, uint32_t seq, int lane) {
    const RingPos rp = ring_pos(seq, R.nslot);
    const uint32_t got = R.got + 4u * rp.slot;
    if (seq >= R.nslot) {
        uint32_t v;
        do { asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(got) : "memory"); } while (v + R.nslot < seq + 1u);
    }
    mbar_wait(R.bar_full + 8u * rp.slot, rp.parity);
    if (lane == 0) asm volatile("st.volatile.shared.u32 [%0], %1;" :: "r"(got), "r"(seq + 1u) : "memory");
    return rp;
}

// ---------------------------------------------------------------- producer warp
__device__ __forceinline__ void producer(const DevProg& P, const DevStage* stages, const DevLin* lins, const uint32_t* s_info,
                                         int cta, int lane, const Ring& R, uint32_t bar_go) {
    uint32_t seq = 0;
    for (int p = 0; p < P.n_phases; ++p) {
        const int s = (int)(s_info[p] & INFO_STAGE) - 1;
        if (s < 0) continue;                                 // no stage of this phase runs on this CTA
        const DevStage& st = stages[s];
        const int rank = cta - st.cta_begin;
        const int KB = st.K / TILE_K;                        // 1 KiB pieces per granule
        const int cp = pg_chunk_pieces(KB);
        for (int gi = rank; gi < st.granules; gi += st.cta_count) {
            int l = st.lin_begin;
            for (int j = 1; j < st.n_lin; ++j)
                if (gi >= lins[st.lin_begin + j].gran_begin) l = st.lin_begin + j;
            const int n32 = gi - lins[l].gran_begin;
            const uint8_t* src = lins[l].packed + (size_t)n32 * KB * 1024;      // the granule is one contiguous run
            for (int p0 = 0; p0 < KB; p0 += cp, ++seq) {
                const int np = min(cp, KB - p0);
                if (P.gate && seq == 1) mbar_wait(bar_go, 0);
                const RingPos rp = ring_pos(seq, R.nslot);
                if (seq >= R.nslot) mbar_wait(R.bar_empty + 8u * rp.slot, rp.parity ^ 1u);      // (every round in turn)
                if (lane == 0) {                              // one bulk copy of up to 30 KiB per chunk
                    mbar_arrive_expect_tx(R.bar_full + 8u * rp.slot, (uint32_t)np * 1024u);
                    tma_bulk_g2s(R.base + rp.slot * R.slot_bytes, src + (size_t)p0 * 1024, (uint32_t)np * 1024u,
                                 R.bar_full + 8u * rp.slot);
                }
            }
        }
    }
}

// ---------------------------------------------------------------- fused activation quant (Eq. 4 lines 1-2)
// The quantised activations of a stage are stored in mma B-fragment order,
//   base + ((kq * MTS + mt) * 32 + lane) * 16  holds  a[8 mt + lane/4][64 kq + 16 (lane%4) .. +15],
// either straight into this CTA's shared memory (LOCAL stages: few elements, every CTA of the group quantises all rows
// itself) or into the stage's scratch in global memory (COOPERATIVE stages: row r is quantised once, by CTA r mod c of
// the stage's group, and every CTA of the group then pulls the finished fragments with one bulk copy).
// A TASK is 16 consecutive elements of one row (two 16-byte loads, one 16-byte fragment store).  The rows this CTA
// handles are first, first + step, ... (< M); task f of a round is handled row f / (K/16), elements 16 (f mod K/16)..,
// and thread tid takes tasks tid and tid + 480: consecutive threads read consecutive 32 bytes, and one row or eight
// spread over all threads.  A round holds its rows in registers between the absmax and the quantisation.
template <bool TO_GLOBAL>
__device__ __forceinline__ void quant_rows(const DevProg& P, const DevStage& st, int tid, int first, int step, int mts, uint32_t xq_s,
                                           uint8_t* frag_g, float* alpha_g, float4* s_scale, unsigned* s_rowmax, bool write_out) {
    const int lane = tid & 31;
    const int K = st.K, M = st.M, cpr = K / 16;              // tasks per row
    const uint32_t inv_cpr = st.inv_cpr;                     // f / cpr = umulhi(f, inv_cpr): exact for f * cpr < 2^32
    const int n_owned = first < M ? (M - first + step - 1) / step : 0;
    const int rpr = max(1, (PG_QNB * PG_CONSUMERS) / cpr);   // rows per round
    for (int j0 = 0; j0 < n_owned; j0 += rpr) {
        const int nt = min(rpr, n_owned - j0) * cpr;
        uint4 v[2 * PG_QNB];
#pragma unroll
        for (int i = 0; i < PG_QNB; ++i) {
            const int f = tid + i * PG_CONSUMERS;
            const int j = (int)__umulhi((uint32_t)f, inv_cpr), c = f - j * cpr;
            const int row = first + (j0 + j) * step;
            const bool ok = f < nt;
            const uint4* src = st.x + ((size_t)row * K) / 8 + c * 2;
            v[2 * i] = ok ? __ldcg(src) : make_uint4(0, 0, 0, 0);
            v[2 * i + 1] = ok ? __ldcg(src + 1) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int i = 0; i < PG_QNB; ++i) {
            const int f = tid + i * PG_CONSUMERS;
            if (f - lane < nt) {                              // (warp-uniform)
                const int row = first + (j0 + (int)__umulhi((uint32_t)f, inv_cpr)) * step;
                const uint32_t m2 = absmax8_packed(v[2 * i + 1], absmax8_packed(v[2 * i], 0u));
                const uint32_t mine = max(m2 & 0xFFFFu, m2 >> 16) << 16;      // fp32 bits of the task's absmax
                const int row_first = __shfl_sync(0xFFFFFFFFu, row, 0), row_last = __shfl_sync(0xFFFFFFFFu, row, 31);
                if (row_first == row_last) {                  // the usual case: the warp's 32 tasks are in one row
                    const uint32_t mw = __reduce_max_sync(0xFFFFFFFFu, mine);
                    if (lane == 0) atomicMax(s_rowmax + row, mw);
                } else if (f < nt) {
                    atomicMax(s_rowmax + row, mine);
                }
            }
        }
        consumer_bar();
        if (tid < 16) {                                      // per row: alpha_m and the bracketing reciprocals
            const float alpha = alpha_of(__uint_as_float(s_rowmax[tid]));
            s_scale[tid] = quant_scales_of_alpha(alpha);
            const int j = (tid - first) / step;              // is row tid one of this round's rows?
            if (tid >= first && tid < M && (tid - first) % step == 0 && j >= j0 && j < j0 + rpr) {
                if (TO_GLOBAL) alpha_g[tid] = alpha;
                if (write_out && st.xs_out) st.xs_out[tid] = alpha;
            }
        }
        consumer_bar();
#pragma unroll
        for (int i = 0; i < PG_QNB; ++i) {
            const int f = tid + i * PG_CONSUMERS;
            if (f < nt) {
                const int j = (int)__umulhi((uint32_t)f, inv_cpr), c = f - j * cpr;
                const int row = first + (j0 + j) * step;
                const uint32_t off = (uint32_t)((((c >> 2) * mts + (row >> 3)) * 32 + (row & 7) * 4 + (c & 3)) * 16);
                const uint4 q = quant16(v[2 * i], v[2 * i + 1], s_scale[row]);
                if (TO_GLOBAL) *reinterpret_cast<uint4*>(frag_g + off) = q;
                else sts128(xq_s + off, q);
                if (write_out && st.xq_out) *reinterpret_cast<uint4*>(st.xq_out + (size_t)row * K + c * 16) = q;
            }
        }
    }
}

// ---------------------------------------------------------------- the MMAs of one warp on one ring chunk
// Blocks lb = first, first + STRIDE, ... (< nb) of the chunk at `slot_addr`; block lb is k block kq0 + lb of the granule.
// The slot goes back to the producer (NARR arrivals on `bar_empty` by this warp) as soon as the warp's last packed words
// are in registers, before their MMAs.
template <int MT, int STRIDE, int GRP, int NARR>
__device__ __forceinline__ void chunk_mma(uint32_t slot_addr, uint32_t bar_empty, uint32_t xq_s, int first, int nb, int kq0,
                                          int lane, int (&acc)[2][MT][4], int (&acc2)[2][4]) {
    const uint32_t wl = slot_addr + (uint32_t)lane * 16u, xl = xq_s + (uint32_t)lane * 16u;
    int lb0 = first;
    do {
        uint4 wv[GRP], xb[GRP], xh[MT == 2 ? GRP : 1];
#pragma unroll
        for (int ii = 0; ii < GRP; ++ii) {
            const int lb = lb0 + ii * STRIDE;
            const bool ok = lb < nb;
            wv[ii] = ok ? lds128(wl + (uint32_t)lb * 512u) : make_uint4(0, 0, 0, 0);
            xb[ii] = ok ? lds128(xl + (uint32_t)((kq0 + lb) * MT) * 512u) : make_uint4(0, 0, 0, 0);
            if (MT == 2) xh[ii] = ok ? lds128(xl + (uint32_t)((kq0 + lb) * MT + 1) * 512u) : make_uint4(0, 0, 0, 0);
        }
        if (lb0 + GRP * STRIDE >= nb) {                       // the last loads of this chunk are out
            __syncwarp();
            if (lane < NARR) mbar_arrive(bar_empty);
        }
#pragma unroll
        for (int ii = 0; ii < GRP; ++ii) {
            if (lb0 + ii * STRIDE < nb) {
                const uint32_t w4[4] = {wv[ii].x, wv[ii].y, wv[ii].z, wv[ii].w};
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const uint32_t wa = w4[2 * c], wb = w4[2 * c + 1];     // channels 16c+g and 16c+g+8
                    const uint32_t a0 = decode64<0>(wa), a1 = decode64<0>(wb), a2 = decode64<1>(wa), a3 = decode64<1>(wb);
                    const uint32_t e0 = decode64<2>(wa), e1 = decode64<2>(wb), e2 = decode64<3>(wa), e3 = decode64<3>(wb);
                    mma_m16n8k32_s8_nv(acc[c][0], a0, a1, a2, a3, xb[ii].x, xb[ii].y);
                    mma_m16n8k32_s8_nv(acc2[c], e0, e1, e2, e3, xb[ii].z, xb[ii].w);
                    if (MT == 2) {
                        mma_m16n8k32_s8_nv(acc[c][1], a0, a1, a2, a3, xh[MT == 2 ? ii : 0].x, xh[MT == 2 ? ii : 0].y);
                        mma_m16n8k32_s8_nv(acc[c][1], e0, e1, e2, e3, xh[MT == 2 ? ii : 0].z, xh[MT == 2 ? ii : 0].w);
                    }
                }
            }
        }
        lb0 += GRP * STRIDE;
    } while (lb0 < nb);
}

template <int MT>
__device__ __forceinline__ void zero_acc(int (&acc)[2][MT][4], int (&acc2)[2][4]) {
#pragma unroll
    for (int c = 0; c < 2; ++c) {
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[c][mt][i] = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) acc2[c][i] = 0;
    }
}
// the warp's partial sums of a granule -> the int32 tile at `rb` ([16 tokens][PG_RED_STRIDE])
template <int MT>
__device__ __forceinline__ void add_to_tile(uint32_t rb, int g, int t, int (&acc)[2][MT][4], int (&acc2)[2][4]) {
#pragma unroll
    for (int c = 0; c < 2; ++c) {
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[c][0][i] += acc2[c][i];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            const uint32_t row0 = rb + (uint32_t)((mt * 8 + 2 * t) * PG_RED_STRIDE + 16 * c + g) * 4u;
            red_shared_add(row0, acc[c][mt][0]);
            red_shared_add(row0 + PG_RED_STRIDE * 4, acc[c][mt][1]);
            red_shared_add(row0 + 8 * 4, acc[c][mt][2]);
            red_shared_add(row0 + (PG_RED_STRIDE + 8) * 4, acc[c][mt][3]);
        }
    }
}
// one output of a finished tile: read the cell, leave zero behind, dequant (Eq. 4 line 3), store
__device__ __forceinline__ void emit(uint32_t rb, int tok, int ech, const DevLin& L, int n32, float alpha, float beta) {
    const uint32_t cell = rb + (uint32_t)(tok * PG_RED_STRIDE + ech) * 4u;
    const int sum = lds32(cell);
    sts32(cell, 0);                                           // the tile is all zero again for its next granule
    const int a = sum >> 6;                                   // the decode's factor 64 leaves exactly
    const size_t o = (size_t)tok * L.N + (size_t)n32 * BLK_N + ech;
    if (L.dtype == 2) {
        reinterpret_cast<int*>(L.out)[o] = a;
    } else {
        const float y = dequant(a, __fmul_rn(alpha, beta));
        if (L.dtype == 0) reinterpret_cast<float*>(L.out)[o] = y;
        else reinterpret_cast<__nv_bfloat16*>(L.out)[o] = __float2bfloat16_rn(y);
    }
}
__device__ __forceinline__ int lin_of(const DevLin* lins, const DevStage& st, int gi) {
    int l = st.lin_begin;
    for (int j = 1; j < st.n_lin; ++j)
        if (gi >= lins[st.lin_begin + j].gran_begin) l = st.lin_begin + j;
    return l;
}

// ---------------------------------------------------------------- a stage on all 15 warps (fewer than 3 granules per CTA)
// rank / G: rank and size of the stage's CTA group.  Warp w takes the k blocks w, w + 15, ... of every chunk.
template <int MT>
__device__ __forceinline__ void stage_gemm(const DevLin* lins, const DevStage& st, int rank, int G, int tid, const Ring& R,
                                           uint32_t red, uint32_t xq_s, const float* s_beta, const float4* s_scale,
                                           uint32_t& seq, uint32_t& gcount) {
    // w through a shuffle: the compiler then knows it is warp-uniform
    const int w = __shfl_sync(0xFFFFFFFFu, tid >> 5, 0), lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int KB = st.K / TILE_K, cp = pg_chunk_pieces(KB), nout = st.M * 32;
    for (int gi = rank; gi < st.granules; gi += G) {
        const int l = lin_of(lins, st, gi);
        const DevLin& L = lins[l];
        const int n32 = gi - L.gran_begin;
        const float beta = s_beta[l - st.lin_begin];          // staged once per stage
        int acc[2][MT][4], acc2[2][4];                        // acc2: second IMMA chain of token tile 0 (ILP)
        zero_acc<MT>(acc, acc2);
        for (int p0 = 0; p0 < KB; p0 += cp, ++seq) {
            const int np = min(cp, KB - p0);
            const RingPos rp = ring_wait(R, seq, lane);
            chunk_mma<MT, PG_W, 2, 1>(R.base + rp.slot * R.slot_bytes, R.bar_empty + 8u * rp.slot, xq_s, w, 2 * np, 2 * p0,
                                      lane, acc, acc2);       // 15 arrivals (one per warp) hand the slot back
        }
        // The 15 per-warp partial sums of an output are added into one int32 tile (two tiles by granule parity: the
        // epilogue of granule g reads and re-zeroes tile g & 1 while the faster warps already add granule g+1 into the other).
        const uint32_t rb = red + (uint32_t)(gcount & 1) * (PG_RED_BUF_INTS * 4);
        add_to_tile<MT>(rb, g, t, acc, acc2);
        consumer_bar();
        for (int idx = tid; idx < nout; idx += PG_CONSUMERS) emit(rb, idx >> 5, idx & 31, L, n32, s_scale[idx >> 5].x, beta);
        ++gcount;
    }
}

// ---------------------------------------------------------------- a stage on three teams of five warps
// Team q takes the CTA's granules n = q, q+3, ... of the stage (ring chunks n * nchunks ..), its warp j the k blocks
// j, j + 5, ... of every chunk.  Against the 15-way split a warp runs three times as many blocks per mbarrier wait /
// reduction / barrier / epilogue, and the teams are in different phases of their granules instead of in lockstep.
template <int MT>
__device__ __forceinline__ void stage_gemm_teams(const DevLin* lins, const DevStage& st, int rank, int G, int tid, const Ring& R,
                                                 uint32_t red, uint32_t xq_s, const float* s_beta, const float4* s_scale,
                                                 uint32_t& seq, uint32_t& gcount) {
    const int w = __shfl_sync(0xFFFFFFFFu, tid >> 5, 0), lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int team = w / PG_TW, j = w - team * PG_TW, ttid = tid - team * (PG_TW * 32);
    const int KB = st.K / TILE_K, cp = pg_chunk_pieces(KB), nch = pg_chunks(KB), nout = st.M * 32;
    const int ng = rank < st.granules ? (st.granules - rank + G - 1) / G : 0;      // this CTA's granules of the stage
    const uint32_t tiles = red + (uint32_t)team * (2 * PG_RED_BUF_INTS * 4);
    uint32_t tpar = 0;
    for (int n = team; n < ng; n += PG_TEAMS) {
        const int gi = rank + n * G;
        const int l = lin_of(lins, st, gi);
        const DevLin& L = lins[l];
        const int n32 = gi - L.gran_begin;
        const float beta = s_beta[l - st.lin_begin];
        int acc[2][MT][4], acc2[2][4];
        zero_acc<MT>(acc, acc2);
        uint32_t cs = seq + (uint32_t)(n * nch);             // ring chunks n * nch .. of this stage
        for (int p0 = 0; p0 < KB; p0 += cp, ++cs) {
            const int np = min(cp, KB - p0);
            const RingPos rp = ring_wait(R, cs, lane);
            chunk_mma<MT, PG_TW, 3, PG_TEAMS>(R.base + rp.slot * R.slot_bytes, R.bar_empty + 8u * rp.slot, xq_s, j, 2 * np,
                                              2 * p0, lane, acc, acc2);       // (the empty barrier counts 15: three arrivals per team warp)
        }
        const uint32_t rb = tiles + tpar * (PG_RED_BUF_INTS * 4);
        add_to_tile<MT>(rb, g, t, acc, acc2);
        team_bar(team);
        for (int idx = ttid; idx < nout; idx += PG_TW * 32) emit(rb, idx >> 5, idx & 31, L, n32, s_scale[idx >> 5].x, beta);
        tpar ^= 1u;
    }
    seq += (uint32_t)(ng * nch);
    gcount += (uint32_t)ng;
}

// ---------------------------------------------------------------- the kernel
// MAXMT = 1: every stage has M <= 8;  MAXMT = 2: M <= 16 (two token tiles).
template <int MAXMT>
__global__ void __launch_bounds__(PG_THREADS, 1) program_kernel(const __grid_constant__ DevProg P) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 127u) & ~127u;
    uint8_t* base_ptr = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t bar_full = base + PG_OFF_BAR, bar_empty = bar_full + 8u * PG_NSLOT_MAX, bar_go = bar_empty + 8u * PG_NSLOT_MAX;
    const uint32_t bar_xq = bar_go + 8u;
    float4* s_scale = reinterpret_cast<float4*>(base_ptr + PG_OFF_ALPHA);
    float* s_beta = reinterpret_cast<float*>(base_ptr + PG_OFF_BETA);
    unsigned* s_rowmax = reinterpret_cast<unsigned*>(base_ptr + PG_OFF_ROWMAX);
    unsigned* s_misc = reinterpret_cast<unsigned*>(base_ptr + PG_OFF_MISC);
    int* red_ptr = reinterpret_cast<int*>(base_ptr + PG_OFF_RED);
    const uint32_t red = base + PG_OFF_RED;
    uint32_t* s_info = reinterpret_cast<uint32_t*>(base_ptr + PG_OFF_INFO);        // per PHASE: this CTA's stage + 1, publish bit
    uint8_t* desc = base_ptr + pg_off_desc(P.n_stages);
    const uint32_t xq_s = base + (uint32_t)pg_off_xq(P.n_stages, P.n_lin);

    const int tid = threadIdx.x, cta = blockIdx.x, G = gridDim.x;
    PG_STAMP(0);
    if (tid == 0) {
        for (int s = 0; s < PG_NSLOT_MAX; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, PG_W);
        }
        mbar_init(bar_go, 1);
        mbar_init(bar_xq, 1);
        fence_barrier_init();
        s_misc[0] = 0u;
        s_misc[1] = 0u;
        for (int sl = 0; sl < PG_NSLOT_MAX; ++sl) reinterpret_cast<volatile unsigned*>(base_ptr + PG_OFF_GOT)[sl] = 0u;
    }
    if (tid < 16) s_rowmax[tid] = 0u;
    for (int i = tid; i < P.n_phases; i += PG_THREADS) s_info[i] = 0u;
    for (int i = tid; i < PG_RED_INTS; i += PG_THREADS) red_ptr[i] = 0;  // accumulation tiles start at zero
    // descriptor tables -> shared memory (they are read on every granule by producer and consumers)
    const int stage_words = P.n_stages * (int)(sizeof(DevStage) / 8), lin_words = P.n_lin * (int)(sizeof(DevLin) / 8);
    {
        const uint2* gs = reinterpret_cast<const uint2*>(P.stages);
        const uint2* gl = reinterpret_cast<const uint2*>(P.lins);
        uint2* d = reinterpret_cast<uint2*>(desc);
        for (int i = tid; i < stage_words; i += PG_THREADS) d[i] = gs[i];
        for (int i = tid; i < lin_words; i += PG_THREADS) d[stage_words + i] = gl[i];
    }
    __syncthreads();
    const DevStage* stages = reinterpret_cast<const DevStage*>(desc);
    const DevLin* lins = reinterpret_cast<const DevLin*>(desc + (size_t)stage_words * 8);
    // Digest of the stage table for this CTA: the groups of one phase are disjoint, so a CTA runs at most one stage per
    // phase; s_info[phase] = that stage + 1 (0: none), plus the phase's publish bit.
    for (int s = tid; s < P.n_stages; s += PG_THREADS) {
        const DevStage& st = stages[s];
        const int rank = cta - st.cta_begin;
        if (st.flags & 2) atomicOr(s_info + st.phase, INFO_PUBLISH);
        if (rank >= 0 && rank < st.cta_count) {
            atomicOr(s_info + st.phase, (uint32_t)(s + 1));
            atomicMax(s_misc, (unsigned)pg_xq_bytes(st.M, st.K));      // this CTA's largest activation matrix
            atomicMax(s_misc + 1, (unsigned)pg_slot_bytes(st.K));      // and largest ring chunk
        }
    }
    __syncthreads();
    // the ring takes what the descriptors and this CTA's quantised activations leave free, in slots of its largest chunk
    Ring R;
    R.base = xq_s + ((s_misc[0] + 127u) & ~127u);
    R.slot_bytes = max(s_misc[1], 1024u);
    R.nslot = min((uint32_t)PG_NSLOT_MAX, (base + (uint32_t)P.smem_bytes - R.base) / R.slot_bytes);
    R.bar_full = bar_full;
    R.bar_empty = bar_empty;
    R.got = base + PG_OFF_GOT;

    if (tid >= PG_CONSUMERS) {
        // Weights never depend on the previous kernel on the stream: the ring starts filling under its tail.
        pdl_launch_dependents();
        producer(P, stages, lins, s_info, cta, tid & 31, R, bar_go);
        return;
    }
    // Programmatic dependent launch: everything above (barrier init, the static descriptor tables, the first ring
    // chunks) may overlap the tail of the previous kernel on this stream; counters, activations and outputs come after.
    pdl_wait();
    // Trigger the next launch NOW: its CTAs take this SM as soon as this CTA exits and run their own prologue (up to their
    // griddepcontrol.wait, which still waits for this whole grid and its memory) under the tail of this grid.
    pdl_launch_dependents();
    PG_STAMP(1);

    bool go_sent = false;
    uint32_t seq = 0, gcount = 0, xq_par = 0;
    unsigned done_prev = 0xFFFFFFFFu;                        // thread 0: what its early arrival on `done` returned
    for (int p = 0; p < P.n_phases; ++p) {
        const uint32_t info = s_info[p];
        const int s = (int)(info & INFO_STAGE) - 1;
        if (s >= 0) {                                        // this CTA runs stage s in phase p
            const DevStage& st = stages[s];
            const int count = st.cta_count, rank = cta - st.cta_begin;
            if (p > 0) {                                     // a phase starts only after every earlier phase has completed
                                                              // (vla_ternary.h: x of ANY of its stages may be an earlier phase's output)
                if (tid == 0) spin_until(P.bp + (p - 1), (unsigned)G);
                consumer_bar();
            }
            PG_STAMP(2);
            // the stage's scales beta -> shared memory (one L2 round trip per stage instead of one per granule)
            // (loaded now, stored after the quantisation: a cold scale costs a DRAM round trip that must not delay this
            // warp's activation loads)
            float beta_r = 0.0f;
            if (tid >= 32 && tid < 32 + st.n_lin) {
                const DevLin& L = lins[st.lin_begin + tid - 32];
                if (L.dtype != 2) beta_r = __ldcg(L.beta);
            }
            const int mts = (MAXMT == 2 && st.M > 8) ? 2 : 1;
            if (st.coop != nullptr) {
                // cooperative quant: this CTA's rows (rank, rank + count, ...) -> the stage's scratch, then publish
                float* alpha_g = reinterpret_cast<float*>(st.coop + pg_xq_bytes(st.M, st.K));
                quant_rows<true>(P, st, tid, rank, count, mts, 0u, st.coop, alpha_g, s_scale, s_rowmax, true);
                consumer_bar();                              // every fragment store of this CTA precedes the release
                if (tid == 0) {
                    const int mine = rank < st.M ? (st.M - rank + count - 1) / count : 0;
                    if (mine) red_release_gpu(P.cnt + s, (unsigned)mine);
                    spin_until(P.cnt + s, (unsigned)st.M);    // all rows of the stage are in the scratch
                    if (P.n_phases == 1) done_prev = atomicAdd(P.done, 1u);      // (its last counter access: see the end)
                    asm volatile("fence.proxy.async.global;" ::: "memory");     // generic-proxy writes -> the bulk copy's reads
                    const uint32_t bytes = (uint32_t)pg_xq_bytes(st.M, st.K);
                    mbar_arrive_expect_tx(bar_xq, bytes);
                    for (uint32_t o = 0; o < bytes; o += 32768u)
                        tma_bulk_g2s(xq_s + o, st.coop + o, min(32768u, bytes - o), bar_xq);
                    if (!go_sent) mbar_arrive(bar_go);
                }
                go_sent = true;
                mbar_wait(bar_xq, xq_par);
                xq_par ^= 1u;
                if (tid < 16) s_scale[tid].x = __ldcg(alpha_g + tid);
            } else {
                // small stage: every CTA of the group quantises all rows into its own shared memory
                quant_rows<false>(P, st, tid, 0, 1, mts, xq_s, nullptr, nullptr, s_scale, s_rowmax, rank == 0);
                const int cpr = st.K / 16, npad = (8 * mts - st.M) * cpr;      // padding rows are zero fragments
                for (int idx = tid; idx < npad; idx += PG_CONSUMERS) {
                    const int j = (int)__umulhi((uint32_t)idx, st.inv_cpr), c = idx - j * cpr, row = st.M + j;
                    sts128(xq_s + (uint32_t)((((c >> 2) * mts + (row >> 3)) * 32 + (row & 7) * 4 + (c & 3)) * 16), make_uint4(0, 0, 0, 0));
                }
                if (!go_sent) {
                    if (tid == 0) mbar_arrive(bar_go);
                    go_sent = true;
                }
            }
            if (tid >= 32 && tid < 32 + st.n_lin) s_beta[tid - 32] = beta_r;
            consumer_bar();                                  // fragments and scales are complete
            if (tid < 16) s_rowmax[tid] = 0u;                // (the next stage's atomics come after its own barriers)
            PG_STAMP(3);
            const bool teams = prog_team_mode(st.granules, count);
            if (MAXMT == 1 || st.M <= 8) {
                if (teams) stage_gemm_teams<1>(lins, st, rank, count, tid, R, red, xq_s, s_beta, s_scale, seq, gcount);
                else stage_gemm<1>(lins, st, rank, count, tid, R, red, xq_s, s_beta, s_scale, seq, gcount);
            } else {
                if (teams) stage_gemm_teams<MAXMT>(lins, st, rank, count, tid, R, red, xq_s, s_beta, s_scale, seq, gcount);
                else stage_gemm<MAXMT>(lins, st, rank, count, tid, R, red, xq_s, s_beta, s_scale, seq, gcount);
            }
            consumer_bar();                                  // everybody is done with xq_s / s_beta / s_scale of this stage
            PG_STAMP(4);
        }
        if (info & INFO_PUBLISH) {                           // end of a phase that a later phase reads from
            consumer_bar();                                  // every output store of this CTA precedes the release
            if (tid == 0) red_release_gpu(P.bp + p, 1u);
        }
    }
    if (!go_sent && tid == 0) mbar_arrive(bar_go);           // (a CTA without a stage: its producer has nothing to copy)
    PG_STAMP(5);
    // Programs with counters (phases, cooperative stages): the last CTA past its last counter access re-zeroes them, so the
    // next launch needs no memset.  In a single-phase program that access is the CTA's spin on its stage's row count (its
    // own rows were released before): it counted itself there, and the atomic's round trip overlapped the GEMM.
    if ((P.n_phases > 1 || P.n_coop > 0) && tid == 0) {
        const unsigned prev = (done_prev != 0xFFFFFFFFu) ? done_prev : atomicAdd(P.done, 1u);
        if (prev == (unsigned)G - 1u) {                      // every CTA is past its last counter access
            for (int q = 0; q < P.n_stages; ++q) { P.bp[q] = 0u; P.cnt[q] = 0u; }
            *P.done = 0u;                                     // (kernel completion makes these visible to the next launch)
        }
    }
}

int program_threads() { return PG_THREADS; }

cudaError_t program_max_ctas_per_sm(int max_m, int smem_bytes, int* out) {
    cudaError_t e = cudaFuncSetAttribute(max_m <= 8 ? (const void*)program_kernel<1> : (const void*)program_kernel<2>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes + 128);
    if (e != cudaSuccess) return e;
    if (max_m <= 8) return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, program_kernel<1>, PG_THREADS, (size_t)smem_bytes + 128);
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, program_kernel<2>, PG_THREADS, (size_t)smem_bytes + 128);
}

cudaError_t launch_program(const DevProg& prog, int grid, int max_m, cudaStream_t s) {
    // the attribute is per device and cheap to set: no process-wide cache (a process may drive several devices)
    cudaError_t e = cudaFuncSetAttribute(max_m <= 8 ? (const void*)program_kernel<1> : (const void*)program_kernel<2>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, prog.smem_bytes + 128);
    if (e != cudaSuccess) return e;
    count_launch();
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(PG_THREADS);
    cfg.dynamicSmemBytes = (size_t)prog.smem_bytes + 128;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (max_m <= 8) return cudaLaunchKernelEx(&cfg, program_kernel<1>, prog);
    return cudaLaunchKernelEx(&cfg, program_kernel<2>, prog);
}

}  // namespace vla
