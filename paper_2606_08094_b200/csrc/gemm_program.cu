// gemm_program.cu -- persistent "program" kernel for the small-M (M <= 16) regime: ONE launch runs a whole list
// of ternary linears (Eq. 4), independent or chained, e.g. the 30-layer stack of
// BASELINE.json configs[3].  PAPER.md line 56 removes dispatch overhead by persisting graphs; on B200 a launch
// costs ~5000 cycles, more than ten times the HBM time of a 1.6 MB weight tensor, so the whole program is one
// kernel and the only thing that ever waits is data.
//
// Grid: one CTA per SM, 16 warps.
//   warp 15 (producer)   streams this CTA's share of the packed weights of EVERY stage, in program order, through
//                        a 6 x 30 KiB (M <= 16 variant: 4 x 30 KiB) shared-memory ring with cp.async.bulk (TMA) + mbarriers.  It never waits on
//                        activations, so HBM stays busy across stage boundaries and grid barriers.
//   warps 0-14 (consumers) per stage: hold the int8 activations as mma.m16n8k32 B fragments IN REGISTERS (warp w
//                        owns the 64-wide k blocks kq = w mod 15), read packed words from the ring, decode them
//                        in registers (2 ALU ops per 4 weights, common.cuh) into A fragments, accumulate int32,
//                        add the 15 partial sums per output into one shared-memory tile (red.shared.add), and run the dequant
//                        epilogue  y = (float)acc * (alpha_m * beta).
// Work unit: a GRANULE = 32 output channels x all of K of one linear (K/128 contiguous 1 KiB pieces of the packed
// layout).  The stages of one PHASE are independent, so they run CONCURRENTLY on disjoint CTA groups sized by their
// weight bytes (no serialisation between them, and each activation matrix is read by its own group only instead
// of by all 148 SMs); granule gi of a stage goes to CTA (gi mod group size) of its group.
// Activation quant (Eq. 4 lines 1-2): row r of stage s is quantised by ONE owner CTA (absmax over the row, then
// the true-division quantiser of quant.cuh) into global int8 + alpha; counters in global memory order the phases:
//   bp[p] = CTAs that finished phase p   (a dependent stage's row owners wait for bp[p-1] == gridDim.x)
//   b2[s] = rows of stage s quantised    (the stage's group waits for b2[s] == M_s before it loads its B fragments)
// int32 sums are exact in any order, so the
// result is bit-identical to the per-call kernels and to the oracle.
#include <cuda_bf16.h>
#include "common.cuh"
#include "kernels.h"
#include "program.h"
#include "quant.cuh"

namespace vla {

// 15 consumer warps + 1 producer = 16 warps = 4 per SM sub-partition -> 128 registers per thread.  (A 17th warp puts
// five warps on one sub-partition and caps every thread at 96 registers: the B fragments then spill, and with 227 KB
// of shared memory there is no L1 to catch the spills.)
constexpr int PG_W = 15;                         // consumer warps
constexpr int PG_CONSUMERS = PG_W * 32;          // 480 threads
constexpr int PG_THREADS = PG_CONSUMERS + 32;    // 512
constexpr int PG_BPW = 4;                         // 512-byte blocks per warp per chunk (one mbarrier wait / release)
constexpr int PG_CHUNK_PIECES = PG_W * PG_BPW / 2;   // 30 pieces of 1 KiB = 60 blocks of 32 ch x 64 k: four per warp
constexpr int PG_SLOT_BYTES = PG_CHUNK_PIECES * 1024;
constexpr int PG_XHI_BYTES = 65536;              // M <= 16 variant: B fragments of tokens 8-15 (8 * K bytes, K <= 8192)
__host__ __device__ constexpr int pg_nslot(int maxmt) { return maxmt == 1 ? 6 : 4; }
constexpr int PG_DESC_BYTES = 15360;             // stage + linear descriptors cached in shared memory
constexpr int PG_NBMAX = 9;                      // k blocks per warp per granule: ceil(128 / 15)  ->  K <= 8192
constexpr int PG_NCHUNK = 3;                     // chunks of 60 blocks that cover 128 blocks
constexpr int PG_RED_STRIDE = 36;                // ints per token row: fragment lane (g,t) -> bank 8t + g, conflict-free
constexpr int PG_RED_BUF_INTS = 16 * PG_RED_STRIDE;   // one [16 tokens][32 channels] int32 accumulation tile
constexpr int PG_TEAMS = 3, PG_TW = 5;           // team mode (K <= 2880): three teams of five warps, one granule each
constexpr int PG_TEAM_NBLK = PG_NBMAX * PG_TW;   // 45 k blocks: a team warp still holds its B fragments in 9 x uint4
static_assert(PG_TEAM_NBLK == 45 && PG_TEAMS == 3, "prog_team_mode() in program.h assumes 45 k blocks and 3 teams");
constexpr int PG_RED_INTS = 2 * PG_TEAMS * PG_RED_BUF_INTS;   // two tiles (granule parity) per team: 13 824 B
// Per-CTA digest of the stage table, built in the prologue (before griddepcontrol.wait): one word per stage, so that the
// scans "which rows do I quantise in this phase" and "which stages is my group in" cost one shared-memory load per stage
// instead of ~250 cycles of dependent descriptor loads (12 independent stages: 2 x 1.5 us at the head of every launch).
constexpr int PG_INFO_WORDS = 288;               // >= PG_DESC_BYTES / sizeof(DevStage)
constexpr uint32_t INFO_RANK = 0xFFFFu;          // rank in the stage's CTA group + 1 (0: not a member)
constexpr uint32_t INFO_PHASE_START = 1u << 16;  // first stage of its phase
constexpr uint32_t INFO_PUBLISH = 1u << 17;      // DevStage.flags bit 1
constexpr uint32_t INFO_OWNS_ROW = 1u << 18;     // grid-wide row ownership and this CTA owns a row of the stage
__host__ __device__ constexpr int pg_smem(int maxmt) {
    return pg_nslot(maxmt) * PG_SLOT_BYTES + PG_RED_INTS * 4 + PG_DESC_BYTES + (maxmt == 1 ? 0 : PG_XHI_BYTES) +
           2 * pg_nslot(maxmt) * 8 + 64 + 16 + 64 + PG_INFO_WORDS * 4 + 128;
}

#ifdef VLA_PROG_TRACE
// debug-only (never defined in the product build): per-CTA globaltimer stamps, read back by vla_debug_read_trace
__device__ unsigned long long g_trace[148 * 1024];
__device__ __forceinline__ void trace(int cta, int& n, int tid) {
    if (tid == 0 && n < 1024) {
        unsigned long long t;
#ifdef VLA_PROG_TRACE_CLOCK
        t = (unsigned long long)clock64();               // SM cycles: cheap, per-CTA differences only
#else
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
#endif
        g_trace[blockIdx.x * 1024 + n++] = t;
    }
}
#define QTRACE(k) do { if (threadIdx.x == 0 && g_trace[blockIdx.x * 1024 + 900 + (k)] == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_trace[blockIdx.x * 1024 + 900 + (k)] = t_; } } while (0)
#define TRACE() trace(cta, tr_n, tid)
#define TRARG , tr_n
// launch-to-launch view: stamp k (0 entry, 1 after griddepcontrol.wait, 2 first MMA may start, 3 end) of the last 16
// launches of every CTA; the launch ordinal rides in the header's magic field (debug build only)
__device__ unsigned long long g_pdl[148 * 16 * 8];
__device__ unsigned g_ord;
#define PDLT(k) do { if (threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_pdl[(blockIdx.x * 16 + (P.magic & 15)) * 8 + (k)] = t_; } } while (0)
#define QT(k) do { if (threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_pdl[(blockIdx.x * 16 + (g_ord & 15)) * 8 + (k)] = t_; } } while (0)
#else
#define PDLT(k) do { } while (0)
#define QT(k) do { } while (0)
#define TRACE()
#define QTRACE(k) do { } while (0)
#define TRARG
#endif

__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;" :: "n"(PG_CONSUMERS) : "memory"); }

__device__ __forceinline__ unsigned ld_acquire_gpu(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void spin_until(const unsigned* p, unsigned target) {
    while (ld_acquire_gpu(p) < target) { }
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr) : "memory");
    return r;
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
__device__ __forceinline__ void red_release_gpu(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}

// non-volatile form: the compiler may interleave it with the decode of the next block
__device__ __forceinline__ void mma_m16n8k32_s8_nv(int (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                                   uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// ---------------------------------------------------------------- producer warp
template <int NSLOT>
__device__ __forceinline__ void producer(const DevProg& P, const DevStage* stages, const DevLin* lins, const uint32_t* s_info, int cta,
                                         int lane, uint32_t ring, uint32_t bar_full, uint32_t bar_empty, uint32_t bar_go) {
    // The first chunk goes out at once; the rest of the ring is filled only after this CTA has its own activation row in
    // registers (row owners) or has seen its first quantised activations (the others): otherwise 148 rings (26 MB) are requested in the first microsecond and the
    // few KB of activation rows the quant owners need queue behind them (measured: 2.5-10 us before the first MMA).
    uint32_t slot = 0, round = 0, issued = 0;
    for (int s = 0; s < P.n_stages; ++s) {
        const int rank = (int)(s_info[s] & INFO_RANK) - 1;
        if (rank < 0) continue;                              // another group's stage
        const DevStage& st = stages[s];
        const int KB = st.K / TILE_K;                       // 1 KiB pieces per granule
        for (int gi = rank; gi < st.granules; gi += st.cta_count) {
            int l = st.lin_begin;
            for (int j = 1; j < st.n_lin; ++j)
                if (gi >= lins[st.lin_begin + j].gran_begin) l = st.lin_begin + j;
            const int n32 = gi - lins[l].gran_begin;
            const uint8_t* src = lins[l].packed + (size_t)n32 * KB * 1024;      // the granule is one contiguous run
            for (int p0 = 0; p0 < KB; p0 += PG_CHUNK_PIECES) {
                const int np = min(PG_CHUNK_PIECES, KB - p0);
                if (issued == 1) mbar_wait(bar_go, 0);
                ++issued;
                if (round > 0) mbar_wait(bar_empty + 8u * slot, (round - 1) & 1);
                if (lane == 0) {                              // one bulk copy of up to 15 KiB per chunk
                    mbar_arrive_expect_tx(bar_full + 8u * slot, (uint32_t)np * 1024u);
                    tma_bulk_g2s(ring + slot * PG_SLOT_BYTES, src + (size_t)p0 * 1024, (uint32_t)np * 1024u,
                                 bar_full + 8u * slot);
                }
                if (++slot == NSLOT) { slot = 0; ++round; }
            }
        }
    }
}

// ---------------------------------------------------------------- row-owner activation quant (Eq. 4 lines 1-2)
// All 512 consumer threads of the owner CTA quantise row r of stage st: one pass, the row lives in registers.
__device__ __forceinline__ void quant_row(const DevStage& st, int r, int tid, float* s_max, uint32_t bar_go, bool& go_sent) {
    const int nvec = st.K / 8;                               // uint4 of 8 bf16; K <= 8192 -> nvec <= 1024
    const uint4* xr = st.x + (size_t)r * nvec;
    const uint4 z = make_uint4(0, 0, 0, 0);
    QTRACE(0);
    QT(4);
    const uint4 v0 = (tid < nvec) ? __ldcg(xr + tid) : z;
    const uint4 v1 = (tid + PG_CONSUMERS < nvec) ? __ldcg(xr + tid + PG_CONSUMERS) : z;
    const uint4 v2 = (tid + 2 * PG_CONSUMERS < nvec) ? __ldcg(xr + tid + 2 * PG_CONSUMERS) : z;
    float m = absmax8(v2, absmax8(v1, absmax8(v0, 0.0f)));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
    if ((tid & 31) == 0) s_max[tid >> 5] = m;
    QTRACE(1);
    consumer_bar();
    if (!go_sent) {                                          // the row is in registers: the ring may fill now
        if (tid == 0) mbar_arrive(bar_go);
        go_sent = true;
    }
    QTRACE(2);
    QT(5);
    m = s_max[0];
#pragma unroll
    for (int i = 1; i < PG_W; ++i) m = fmaxf(m, s_max[i]);
    const float alpha = alpha_of(m);
    if (tid == 0) st.xs[r] = alpha;
    uint2* qr = st.xq + (size_t)r * nvec;
    if (tid < nvec) qr[tid] = quant8(v0, alpha);
    if (tid + PG_CONSUMERS < nvec) qr[tid + PG_CONSUMERS] = quant8(v1, alpha);
    if (tid + 2 * PG_CONSUMERS < nvec) qr[tid + 2 * PG_CONSUMERS] = quant8(v2, alpha);
    QTRACE(3);
    consumer_bar();                                          // s_max may be reused; stores precede thread 0's fence
    QTRACE(4);
    QT(6);
}

// Row r of stage s is quantised by CTA (row_begin_s + r) mod gridDim.x (row_begin_s is stored reduced mod gridDim.x) -- any CTA, not only the stage's group, so that
// the rows of all stages of a phase are spread over the whole grid (a 2-CTA group would otherwise quantise 8 rows
// one after the other).  Called by every CTA at the start of a phase, for all stages [s0, s1) of the phase.
// own_stage = true: only stage s0, and only if its rows stay inside its group (flag bit 2).
__device__ __forceinline__ void quant_phase_rows(const DevProg& P, const DevStage* stages, const uint32_t* s_info, int s0,
                                                 int cta, int G, int tid, float* s_max, bool own_stage, uint32_t bar_go, bool& go_sent) {
    const int phase = stages[s0].phase;
    bool waited = false;
    for (int s = s0; s < (own_stage ? s0 + 1 : P.n_stages) && (s == s0 || !(s_info[s] & INFO_PHASE_START)); ++s) {
        if (!own_stage && !(s_info[s] & INFO_OWNS_ROW)) continue;        // nothing of this stage is mine (one load)
        const DevStage& st = stages[s];
        int r, step;
        if (st.flags & 4) {                                   // rows stay inside the stage's own CTA group
            if (!own_stage) continue;                         // (quantised when the group reaches the stage)
            r = cta - st.cta_begin;
            step = st.cta_count;
            if (r < 0 || r >= step) continue;
        } else {                                              // first row with (row_begin + r) % G == cta
            if (own_stage) continue;
            r = cta - st.row_begin;                           // row_begin is already reduced mod gridDim.x
            if (r < 0) r += G;
            step = G;
        }
        unsigned done_rows = 0;
        for (; r < st.M; r += step, ++done_rows) {
            if (phase > 0 && !waited) {                       // a phase starts only after every earlier phase has completed
                                                              // (vla_ternary.h: x of ANY of its stages may be an earlier phase's output)
                if (tid == 0) spin_until(P.bp + (phase - 1), (unsigned)G);
                consumer_bar();
                waited = true;
            }
            quant_row(st, r, tid, s_max, bar_go, go_sent);
        }
        if (done_rows != 0 && tid == 0) red_release_gpu(P.b2 + s, done_rows);    // one release per stage
        if (done_rows != 0) QT(7);
    }
}

// ---------------------------------------------------------------- one stage's granules on the consumer warps
// int8 activations of this warp's k blocks (kq = 16 i + w), as mma B fragments, in registers for the whole stage
// Tokens 0-7 stay in registers (xv); in the M <= 16 variant the fragments of tokens 8-15 go to this thread's private
// 16-byte slots of the shared-memory region xhi (64 registers of fragments would spill, and with 227 KB of shared
// memory there is no L1 left to catch spills).
__device__ __forceinline__ void sts128(uint32_t addr, uint4 v) {
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" :: "r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
template <int MAXMT, int W>
__device__ __forceinline__ void load_xv(const DevStage& st, int tid, uint4 (&xv)[PG_NBMAX], uint32_t xhi) {
    const int w = (tid >> 5) % W, lane = tid & 31, g = lane >> 2, t = lane & 3;   // W = 5: the warp's index in its team
    const int K = st.K, nblk = K / BLK_K;
    const int8_t* xq = reinterpret_cast<const int8_t*>(st.xq);
    // all loads first, then the shared-memory stores: sts128 is a compiler barrier, and a load issued after it would
    // wait for the previous one (measured: 9 serial L2 round trips = 3.7 us at M = 16)
    uint4 hi[MAXMT == 1 ? 1 : PG_NBMAX];
#pragma unroll
    for (int i = 0; i < PG_NBMAX; ++i)
#pragma unroll
        for (int mt = 0; mt < MAXMT; ++mt) {
            const int kq = i * W + w, tok = mt * 8 + g;
            const uint4 v = (kq < nblk && tok < st.M)
                                ? __ldcg(reinterpret_cast<const uint4*>(xq + (size_t)tok * K + kq * BLK_K + t * 16))
                                : make_uint4(0, 0, 0, 0);
            if (mt == 0) xv[i] = v;
            else hi[i] = v;
        }
    if (MAXMT == 2) {
#pragma unroll
        for (int i = 0; i < PG_NBMAX; ++i) {
            const int kq = i * W + w;
            if (kq < nblk) sts128(xhi + (uint32_t)(kq * 32 + lane) * 16u, hi[MAXMT == 1 ? 0 : i]);
        }
    }
}

// cta / G: rank and size of the stage's CTA group
template <int MT, int NSLOT>
__device__ __forceinline__ void stage_gemm(const DevLin* lins, const DevStage& st, int cta, int G,
                                           int tid, uint32_t ring, int* red, const float* s_beta, uint32_t bar_full, uint32_t bar_empty,
                                           uint4 (&xv)[PG_NBMAX], uint32_t xhi, uint32_t& slot, uint32_t& phase, uint32_t& gcount
#ifdef VLA_PROG_TRACE
                                           , int& tr_n
#endif
                                           ) {
    constexpr int MTOK = MT * 8;
    // w through a shuffle: the compiler then knows it is warp-uniform and the per-block range checks below become
    // uniform branches (no BSSY/BSYNC reconvergence around every block)
    const int w = __shfl_sync(0xFFFFFFFFu, tid >> 5, 0), lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int M = st.M, nblk = st.K / BLK_K, KB = st.K / TILE_K;
    const int nchunks = (KB + PG_CHUNK_PIECES - 1) / PG_CHUNK_PIECES;
    // epilogue role: output (token tid/32, channel tid%32); the 32 threads of warp 0 also take token 15
    const int etok = tid >> 5, ech = tid & 31;
    const bool eactive = (etok < M) && (etok < MTOK);
    const bool eactive2 = (MT == 2) && (tid < 32) && (M == 16);
    const float alpha = eactive ? __ldcg(st.xs + etok) : 0.0f;
    const float alpha2 = eactive2 ? __ldcg(st.xs + 15) : 0.0f;
    const uint32_t my_off = (uint32_t)(w * 512 + lane * 16);  // block b = ii*15 + w of the chunk

    for (int gi = cta; gi < st.granules; gi += G) {
        TRACE();
        int l = st.lin_begin;
        for (int j = 1; j < st.n_lin; ++j)
            if (gi >= lins[st.lin_begin + j].gran_begin) l = st.lin_begin + j;
        const DevLin& L = lins[l];
        const int n32 = gi - L.gran_begin;
        const float beta = s_beta[l - st.lin_begin];          // staged once per stage

#ifdef VLA_PROG_TRACE
        long long twait = 0;
#endif
        int acc[2][MT][4], acc2[2][4];                        // acc2: second IMMA chain of token tile 0 (ILP)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int i = 0; i < 4; ++i) acc[c][mt][i] = 0;
#pragma unroll
            for (int i = 0; i < 4; ++i) acc2[c][i] = 0;
        }

#pragma unroll
        for (int ck = 0; ck < PG_NCHUNK; ++ck) {              // 3 chunks of 30 KiB cover K <= 8192
            if (ck < nchunks) {
#ifdef VLA_PROG_TRACE
                long long tw0 = clock64();
#endif
                mbar_wait(bar_full + 8u * slot, phase);
#ifdef VLA_PROG_TRACE
                twait += clock64() - tw0;
#endif
                // the four blocks of this warp in the chunk, two at a time; the slot is handed back once the last two
                // are in registers
#pragma unroll
                for (int half = 0; half < PG_BPW / 2; ++half) {
                    uint4 wv[2];
#pragma unroll
                    for (int ii = 0; ii < 2; ++ii) {
                        const int i = PG_BPW * ck + 2 * half + ii;
                        wv[ii] = (i < PG_NBMAX && i * PG_W + w < nblk)
                                     ? lds128(ring + slot * PG_SLOT_BYTES + (2 * half + ii) * (PG_W * 512) + my_off)
                                     : make_uint4(0, 0, 0, 0);
                    }
                    if (half == PG_BPW / 2 - 1) {
                        __syncwarp();
                        if (lane == 0) mbar_arrive(bar_empty + 8u * slot);   // release: ordered after the loads above
                    }
#pragma unroll
                    for (int ii = 0; ii < 2; ++ii) {
                        const int i = PG_BPW * ck + 2 * half + ii;
                        if (i < PG_NBMAX && i * PG_W + w < nblk) {
                            const uint32_t w4[4] = {wv[ii].x, wv[ii].y, wv[ii].z, wv[ii].w};
                            uint4 xh = make_uint4(0, 0, 0, 0);    // tokens 8-15 of this block (M <= 16 variant)
                            if (MT == 2) xh = lds128(xhi + (uint32_t)((i * PG_W + w) * 32 + lane) * 16u);
#pragma unroll
                            for (int c = 0; c < 2; ++c) {
                                const uint32_t wa = w4[2 * c], wb = w4[2 * c + 1];     // channels 16c+g and 16c+g+8
                                const uint32_t a0 = decode64<0>(wa), a1 = decode64<0>(wb), a2 = decode64<1>(wa), a3 = decode64<1>(wb);
                                const uint32_t e0 = decode64<2>(wa), e1 = decode64<2>(wb), e2 = decode64<3>(wa), e3 = decode64<3>(wb);
                                mma_m16n8k32_s8_nv(acc[c][0], a0, a1, a2, a3, xv[i < PG_NBMAX ? i : 0].x, xv[i < PG_NBMAX ? i : 0].y);
                                mma_m16n8k32_s8_nv(acc2[c], e0, e1, e2, e3, xv[i < PG_NBMAX ? i : 0].z, xv[i < PG_NBMAX ? i : 0].w);
                                if (MT == 2) {
                                    mma_m16n8k32_s8_nv(acc[c][1], a0, a1, a2, a3, xh.x, xh.y);
                                    mma_m16n8k32_s8_nv(acc[c][1], e0, e1, e2, e3, xh.z, xh.w);
                                }
                            }
                        }
                    }
                }
                if (++slot == NSLOT) { slot = 0; phase ^= 1; }
            }
        }

#ifdef VLA_PROG_TRACE
        if (tid == 0 && tr_n < 1024) g_trace[blockIdx.x * 1024 + tr_n++] = (unsigned long long)twait;   // cycles, not a stamp
#endif
        TRACE();
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[c][0][i] += acc2[c][i];
        // The 15 per-warp partial sums of an output are added into one int32 tile in shared memory (red.shared.add:
        // integer addition is exact in any order), two tiles by granule parity: the epilogue of granule g reads and
        // re-zeroes tile g & 1 while the faster warps already add granule g+1 into the other one.
        const uint32_t rb = smem_u32(red) + (uint32_t)(gcount & 1) * (PG_RED_BUF_INTS * 4);
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const uint32_t row0 = rb + (uint32_t)((mt * 8 + 2 * t) * PG_RED_STRIDE + 16 * c + g) * 4u;
                red_shared_add(row0, acc[c][mt][0]);
                red_shared_add(row0 + PG_RED_STRIDE * 4, acc[c][mt][1]);
                red_shared_add(row0 + 8 * 4, acc[c][mt][2]);
                red_shared_add(row0 + (PG_RED_STRIDE + 8) * 4, acc[c][mt][3]);
            }
        consumer_bar();
        TRACE();
#pragma unroll
        for (int rep = 0; rep < MT; ++rep) {
            const bool act = rep == 0 ? eactive : eactive2;
            const int tok = rep == 0 ? etok : 15;
            if (act) {
                const uint32_t cell = rb + (uint32_t)(tok * PG_RED_STRIDE + ech) * 4u;
                const int sum = lds32(cell);
                sts32(cell, 0);                               // the tile is all zero again for granule g+2
                const int a = sum >> 6;                       // the decode's factor 64 leaves exactly
                const size_t o = (size_t)tok * L.N + (size_t)n32 * BLK_N + ech;
                if (L.dtype == 2) {
                    reinterpret_cast<int*>(L.out)[o] = a;
                } else {
                    const float y = dequant(a, __fmul_rn(rep == 0 ? alpha : alpha2, beta));
                    if (L.dtype == 0) reinterpret_cast<float*>(L.out)[o] = y;
                    else reinterpret_cast<__nv_bfloat16*>(L.out)[o] = __float2bfloat16_rn(y);
                }
            }
        }
        TRACE();
        ++gcount;
    }
}

// ---------------------------------------------------------------- team mode (K <= 2880, >= 2 granules per CTA)
// The 15 consumer warps work as THREE independent teams of five: team q takes the CTA's granules n = q, q+3, ... of the
// stage (ring chunk n: with K <= 3840 a chunk is exactly one granule, so the producer is unchanged), its warp j owns the
// k blocks kq = j (mod 5).  Against the 15-way split a warp runs 8 blocks instead of 3 per mbarrier wait / reduction /
// barrier / epilogue, and the three teams are in different phases of their granules instead of in lockstep (chunk
// arrival -> decode burst -> barrier), which is what bounded the 15-way loop.
__device__ __forceinline__ void team_bar(int team) {
    asm volatile("bar.sync %0, %1;" :: "r"(2 + team), "n"(PG_TW * 32) : "memory");
}
template <int MT, int NSLOT>
__device__ __forceinline__ void stage_gemm_teams(const DevLin* lins, const DevStage& st, int rank, int G, int tid, uint32_t ring,
                                                 int* red, const float* s_beta, const float* s_alpha, uint32_t bar_full,
                                                 uint32_t bar_empty, uint4 (&xv)[PG_NBMAX], uint32_t xhi, uint32_t& slot,
                                                 uint32_t& phase, uint32_t& gcount) {
    const int w = __shfl_sync(0xFFFFFFFFu, tid >> 5, 0), lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int team = w / PG_TW, j = w - team * PG_TW, ttid = tid - team * (PG_TW * 32);
    const int nblk = st.K / BLK_K, nout = st.M * 32;
    const int ng = rank < st.granules ? (st.granules - rank + G - 1) / G : 0;      // this CTA's granules (= ring chunks)
    const uint32_t tiles = smem_u32(red) + (uint32_t)team * (2 * PG_RED_BUF_INTS * 4);
    uint32_t tpar = 0;
    for (int n = team; n < ng; n += PG_TEAMS) {
        const int gi = rank + n * G;
        int l = st.lin_begin;
        for (int q = 1; q < st.n_lin; ++q)
            if (gi >= lins[st.lin_begin + q].gran_begin) l = st.lin_begin + q;
        const DevLin& L = lins[l];
        const int n32 = gi - L.gran_begin;
        const float beta = s_beta[l - st.lin_begin];
        uint32_t sl = slot + (uint32_t)n;                     // ring position of chunk n of this stage
        const uint32_t wraps = sl / NSLOT;
        sl -= wraps * NSLOT;
        const uint32_t ph = phase ^ (wraps & 1u);

        int acc[2][MT][4], acc2[2][4];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int i = 0; i < 4; ++i) acc[c][mt][i] = 0;
#pragma unroll
            for (int i = 0; i < 4; ++i) acc2[c][i] = 0;
        }
        mbar_wait(bar_full + 8u * sl, ph);
        const uint32_t src = ring + sl * PG_SLOT_BYTES + (uint32_t)lane * 16u;   // block kq of the granule at kq * 512
#pragma unroll
        for (int i0 = 0; i0 < PG_NBMAX; i0 += 3) {
            uint4 wv[3];
#pragma unroll
            for (int ii = 0; ii < 3; ++ii) {
                const int kq = (i0 + ii) * PG_TW + j;
                wv[ii] = (kq < nblk) ? lds128(src + (uint32_t)kq * 512u) : make_uint4(0, 0, 0, 0);
            }
            if (i0 + 3 >= PG_NBMAX) {                         // last loads are out: hand the slot back
                __syncwarp();                                 // (the empty barrier counts 15: three arrivals per team warp)
                if (lane < PG_TEAMS) mbar_arrive(bar_empty + 8u * sl);
            }
#pragma unroll
            for (int ii = 0; ii < 3; ++ii) {
                const int i = i0 + ii, kq = i * PG_TW + j;
                if (kq < nblk) {
                    const uint32_t w4[4] = {wv[ii].x, wv[ii].y, wv[ii].z, wv[ii].w};
                    uint4 xh = make_uint4(0, 0, 0, 0);
                    if (MT == 2) xh = lds128(xhi + (uint32_t)(kq * 32 + lane) * 16u);
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const uint32_t wa = w4[2 * c], wb = w4[2 * c + 1];
                        const uint32_t a0 = decode64<0>(wa), a1 = decode64<0>(wb), a2 = decode64<1>(wa), a3 = decode64<1>(wb);
                        const uint32_t e0 = decode64<2>(wa), e1 = decode64<2>(wb), e2 = decode64<3>(wa), e3 = decode64<3>(wb);
                        mma_m16n8k32_s8_nv(acc[c][0], a0, a1, a2, a3, xv[i].x, xv[i].y);
                        mma_m16n8k32_s8_nv(acc2[c], e0, e1, e2, e3, xv[i].z, xv[i].w);
                        if (MT == 2) {
                            mma_m16n8k32_s8_nv(acc[c][1], a0, a1, a2, a3, xh.x, xh.y);
                            mma_m16n8k32_s8_nv(acc[c][1], e0, e1, e2, e3, xh.z, xh.w);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[c][0][i] += acc2[c][i];
        const uint32_t rb = tiles + tpar * (PG_RED_BUF_INTS * 4);
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const uint32_t row0 = rb + (uint32_t)((mt * 8 + 2 * t) * PG_RED_STRIDE + 16 * c + g) * 4u;
                red_shared_add(row0, acc[c][mt][0]);
                red_shared_add(row0 + PG_RED_STRIDE * 4, acc[c][mt][1]);
                red_shared_add(row0 + 8 * 4, acc[c][mt][2]);
                red_shared_add(row0 + (PG_RED_STRIDE + 8) * 4, acc[c][mt][3]);
            }
        team_bar(team);
        for (int idx = ttid; idx < nout; idx += PG_TW * 32) {  // one output per thread and pass: token idx / 32, channel idx % 32
            const int tok = idx >> 5, ech = idx & 31;
            const uint32_t cell = rb + (uint32_t)(tok * PG_RED_STRIDE + ech) * 4u;
            const int sum = lds32(cell);
            sts32(cell, 0);
            const int a = sum >> 6;
            const size_t o = (size_t)tok * L.N + (size_t)n32 * BLK_N + ech;
            if (L.dtype == 2) {
                reinterpret_cast<int*>(L.out)[o] = a;
            } else {
                const float y = dequant(a, __fmul_rn(s_alpha[tok], beta));
                if (L.dtype == 0) reinterpret_cast<float*>(L.out)[o] = y;
                else reinterpret_cast<__nv_bfloat16*>(L.out)[o] = __float2bfloat16_rn(y);
            }
        }
        tpar ^= 1u;
    }
    uint32_t sl = slot + (uint32_t)ng;                        // every warp: the ring position after this stage's chunks
    const uint32_t wraps = sl / NSLOT;
    slot = sl - wraps * NSLOT;
    phase ^= (wraps & 1u);
    gcount += (uint32_t)ng;
    consumer_bar();                                           // all three teams are done with s_beta / s_alpha / xhi
}

// ---------------------------------------------------------------- the kernel
// MAXMT = 1: every stage has M <= 8 (32 registers of B fragments per thread, no spills);  MAXMT = 2: M <= 16.
template <int MAXMT>
__global__ void __launch_bounds__(PG_THREADS, 1) program_kernel(const __grid_constant__ DevProg P) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 127u) & ~127u;
    uint8_t* base_ptr = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t ring = base;
    constexpr int NSLOT = pg_nslot(MAXMT);
    constexpr int XHI = (MAXMT == 1) ? 0 : PG_XHI_BYTES;
    int* red = reinterpret_cast<int*>(base_ptr + NSLOT * PG_SLOT_BYTES);
    uint8_t* desc = base_ptr + NSLOT * PG_SLOT_BYTES + PG_RED_INTS * 4;
    const uint32_t xhi = base + NSLOT * PG_SLOT_BYTES + PG_RED_INTS * 4 + PG_DESC_BYTES;
    const uint32_t bar_full = xhi + XHI;
    const uint32_t bar_empty = bar_full + 8u * NSLOT;
    const uint32_t bar_go = bar_empty + 8u * NSLOT + 64u;    // after s_max (64 B)
    float* s_beta = reinterpret_cast<float*>(desc + PG_DESC_BYTES + XHI + 16 * NSLOT + 64 + 16);   // 16 floats
    float* s_max = reinterpret_cast<float*>(desc + PG_DESC_BYTES + XHI + 16 * NSLOT);
    uint32_t* s_info = reinterpret_cast<uint32_t*>(desc + PG_DESC_BYTES + XHI + 16 * NSLOT + 64 + 16 + 64);

    const int tid = threadIdx.x, cta = blockIdx.x, G = gridDim.x;
    PDLT(0);
    if (tid == 0) {
        for (int s = 0; s < NSLOT; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, PG_W);
        }
        mbar_init(bar_go, 1);
        fence_barrier_init();
    }
    for (int i = tid; i < PG_RED_INTS; i += PG_THREADS) red[i] = 0;      // accumulation tiles start at zero
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
    for (int s = tid; s < P.n_stages; s += PG_THREADS) {     // the digest of the stage table for this CTA
        const DevStage& st = reinterpret_cast<const DevStage*>(desc)[s];
        const int rank = cta - st.cta_begin;
        uint32_t info = (rank >= 0 && rank < st.cta_count) ? (uint32_t)(rank + 1) : 0u;
        if (s == 0 || reinterpret_cast<const DevStage*>(desc)[s - 1].phase != st.phase) info |= INFO_PHASE_START;
        if (st.flags & 2) info |= INFO_PUBLISH;
        if (!(st.flags & 4)) {
            int r = cta - st.row_begin;                       // first row with (row_begin + r) % G == cta
            if (r < 0) r += G;
            if (r < st.M) info |= INFO_OWNS_ROW;
        }
        s_info[s] = info;
    }
    __syncthreads();
    // Programmatic dependent launch: everything above (barrier init, the static descriptor tables) may overlap the
    // tail of the previous kernel on this stream; counters, activations, weights-in-flight and outputs come after.
    pdl_wait();
    PDLT(1);
#ifdef VLA_PROG_TRACE
    if (tid == 0) g_ord = P.magic;
#endif
    // Trigger the next launch NOW: its CTAs take this SM as soon as this CTA exits and run their own prologue (up to their
    // griddepcontrol.wait, which still waits for this whole grid and its memory) under the tail of this grid.
    pdl_launch_dependents();
    const DevStage* stages = reinterpret_cast<const DevStage*>(desc);
    const DevLin* lins = reinterpret_cast<const DevLin*>(desc + (size_t)stage_words * 8);

    if (tid >= PG_CONSUMERS) {
        producer<NSLOT>(P, stages, lins, s_info, cta, tid & 31, ring, bar_full, bar_empty, bar_go);
        return;
    }
#ifdef VLA_PROG_TRACE
    int tr_n = 0;
#endif
    TRACE();
    uint4 xv[PG_NBMAX];
    bool go_sent = false;
    uint32_t slot = 0, phase = 0, gcount = 0;
    unsigned done_prev = 0xFFFFFFFFu;                        // thread 0: what its early arrival on `done` returned
    for (int s = 0; s < P.n_stages; ++s) {
        const uint32_t info = s_info[s];
        if (info & INFO_PHASE_START) {                       // a new phase: quantise the rows this CTA owns
            TRACE();
            quant_phase_rows(P, stages, s_info, s, cta, G, tid, s_max, false, bar_go, go_sent);
            TRACE();
        }
        const int rank = (int)(info & INFO_RANK) - 1;
        if (rank >= 0) {                                     // this CTA belongs to the stage's group
            const DevStage& st = stages[s];
            const int count = st.cta_count;
            if (st.flags & 4) quant_phase_rows(P, stages, s_info, s, cta, G, tid, s_max, true, bar_go, go_sent);
            TRACE();
            if (tid == 0) {
                spin_until(P.b2 + s, (unsigned)st.M);
                if (!go_sent) mbar_arrive(bar_go);            // let the producer fill the rest of the ring
                if (P.n_phases == 1) {
                    // Single-phase program (a CTA is in exactly one group): this was the CTA's last access to the program's
                    // counters.  Count it as done NOW: the round trip of the atomic overlaps the stage's GEMM instead of
                    // sitting between the last CTA's last store and the end of the grid (~0.4 us of an 18 us decode step).
                    // Every counter the reset clears has its final value by then: a stage's members pass their spin only
                    // after all of its rows' arrivals, and they count themselves done after that spin (no fence needed).
                    done_prev = atomicAdd(P.done, 1u);
                }
            }
            go_sent = true;
            // the stage's scales beta -> shared memory (one L2 round trip per stage instead of one per granule)
            if (tid >= 32 && tid < 32 + st.n_lin) {
                const DevLin& L = lins[st.lin_begin + tid - 32];
                s_beta[tid - 32] = (L.dtype != 2) ? __ldcg(L.beta) : 0.0f;
            }
            consumer_bar();
            TRACE();
            PDLT(2);
            // team mode: the B fragments of a five-way k split still fit in registers and every team gets >= 2 granules
            const bool teams = prog_team_mode(st.K, st.granules, count);
            if (teams) {
                if (tid < st.M) s_max[tid] = __ldcg(st.xs + tid);     // alpha_m for the team epilogues (s_max is free here)
                load_xv<MAXMT, PG_TW>(st, tid, xv, xhi);
                consumer_bar();                               // s_max and (M > 8) the shared B fragments are complete
                if (MAXMT == 1 || st.M <= 8)
                    stage_gemm_teams<1, NSLOT>(lins, st, rank, count, tid, ring, red, s_beta, s_max, bar_full, bar_empty, xv, xhi, slot, phase, gcount);
                else
                    stage_gemm_teams<MAXMT, NSLOT>(lins, st, rank, count, tid, ring, red, s_beta, s_max, bar_full, bar_empty, xv, xhi, slot, phase, gcount);
            } else {
                load_xv<MAXMT, PG_W>(st, tid, xv, xhi);
                if (MAXMT == 1 || st.M <= 8)
                    stage_gemm<1, NSLOT>(lins, st, rank, count, tid, ring, red, s_beta, bar_full, bar_empty, xv, xhi, slot, phase, gcount TRARG);
                else
                    stage_gemm<MAXMT, NSLOT>(lins, st, rank, count, tid, ring, red, s_beta, bar_full, bar_empty, xv, xhi, slot, phase, gcount TRARG);
            }
            TRACE();
        }
        if (info & INFO_PUBLISH) {                           // end of a phase that a later phase reads from
            consumer_bar();                                  // every output store of this CTA precedes the release
            if (tid == 0) red_release_gpu(P.bp + stages[s].phase, 1u);
            TRACE();
        }
    }
    PDLT(3);
    // the last CTA to finish re-zeroes the counters, so the next launch of the same program needs no memset
    if (tid == 0) {
        const unsigned prev = (done_prev != 0xFFFFFFFFu) ? done_prev : atomicAdd(P.done, 1u);
        if (prev == (unsigned)G - 1u) {                      // every CTA is past its last counter access
            for (int s = 0; s < P.n_stages; ++s) P.b2[s] = 0u;
            for (int q = 0; q < P.n_phases; ++q) P.bp[q] = 0u;
            *P.done = 0u;                                     // (kernel completion makes these visible to the next launch)
        }
    }
}

size_t program_desc_capacity() { return PG_DESC_BYTES; }

cudaError_t launch_program(const DevProg& prog, int grid, int max_m, cudaStream_t s) {
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(program_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, pg_smem(1));
        if (e == cudaSuccess) e = cudaFuncSetAttribute(program_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, pg_smem(2));
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    count_launch();
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(PG_THREADS);
    cfg.dynamicSmemBytes = (size_t)pg_smem(max_m <= 8 ? 1 : 2);
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
#ifdef VLA_PROG_TRACE
    static unsigned trace_launch = 0;
    DevProg h = prog;
    h.magic = trace_launch++;
    if (max_m <= 8) return cudaLaunchKernelEx(&cfg, program_kernel<1>, h);
    return cudaLaunchKernelEx(&cfg, program_kernel<2>, h);
#else
    if (max_m <= 8) return cudaLaunchKernelEx(&cfg, program_kernel<1>, prog);
    return cudaLaunchKernelEx(&cfg, program_kernel<2>, prog);
#endif
}

#ifdef VLA_PROG_TRACE
extern "C" int vla_debug_read_trace(unsigned long long* host, size_t n) {
    return (int)cudaMemcpyFromSymbol(host, g_trace, n * sizeof(unsigned long long));
}
extern "C" int vla_debug_read_pdl(unsigned long long* host, size_t n) {
    return (int)cudaMemcpyFromSymbol(host, g_pdl, n * sizeof(unsigned long long));
}
#endif

}  // namespace vla
