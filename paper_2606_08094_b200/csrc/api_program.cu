// api_program.cu -- host side of the program API of include/vla_ternary.h: validation, compilation of the
// descriptor tables into device memory, and the single launch.  Nothing here computes.
#include "../../include/vla_ternary.h"
#include <cstdio>
#include <cstring>
#include <mutex>
#include <unordered_map>
#include <algorithm>
#include <cmath>
#include <vector>
#include "kernels.h"
#include "program.h"
#include "lprogram.h"
#include "gemm_large.cuh"

// partition model constants (SM cycles; see vla_program_build).  Compile-time defaults, overridable for calibration.
#ifndef VLA_PROG_GATE
#define VLA_PROG_GATE 0
#endif
#ifndef VLA_PG_START0
#define VLA_PG_START0 3300.0
#endif
#ifndef VLA_PG_START1
#define VLA_PG_START1 2.5
#endif
#ifndef VLA_PG_START_COOP
#define VLA_PG_START_COOP 9000.0
#endif
#ifndef VLA_PG_T1A
#define VLA_PG_T1A 200.0
#endif
#ifndef VLA_PG_T1B
#define VLA_PG_T1B 55.0
#endif
#ifndef VLA_PG_T2A
#define VLA_PG_T2A 700.0
#endif
#ifndef VLA_PG_T2B
#define VLA_PG_T2B 75.0
#endif
#ifndef VLA_PG_F1A
#define VLA_PG_F1A 954.0
#endif
#ifndef VLA_PG_F1B
#define VLA_PG_F1B 50.0
#endif
#ifndef VLA_PG_F2A
#define VLA_PG_F2A 1212.0
#endif
#ifndef VLA_PG_F2B
#define VLA_PG_F2B 75.0
#endif

namespace {

using vla::DevLin;
using vla::DevProg;
using vla::DevStage;

struct ProgInfo { int grid; int n_stages; int max_m; DevProg header; bool large; vla::DevLProg lheader; };
std::mutex g_mu;
std::unordered_map<const void*, ProgInfo> g_programs;

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline size_t round256(size_t b) { return (b + 255) / 256 * 256; }

// LARGE programs (every stage has M > 16 tokens): the persistent tcgen05 kernel of gemm_lprog.cu
bool is_large(const vla_prog_stage* st) { return st[0].M > 16; }

vla_status check_large(const vla_prog_stage* st, int n) {
    for (int s = 0; s < n; ++s) {
        const vla_prog_stage& a = st[s];
        if (!a.x_bf16 || !a.linears) return VLA_ERR_NULL;
        if (a.M <= 16 || a.M > 32768 || a.K < 128 || a.K % 128 != 0 || a.K > 8192) return VLA_ERR_SHAPE;
        if (a.n_linears < 1 || a.n_linears > 8) return VLA_ERR_SHAPE;
        if (a.depends < 0 || a.depends > s) return VLA_ERR_SHAPE;         // d >= 1: waits for the stages up to s - d (large programs)
        if (!aligned16(a.x_bf16) || (a.xq_opt && !aligned16(a.xq_opt)) || (a.x_scale_opt && !aligned16(a.x_scale_opt)))
            return VLA_ERR_ALIGN;
        for (int j = 0; j < a.n_linears; ++j) {
            const vla_prog_linear& l = a.linears[j];
            if (l.out_dtype < 0 || l.out_dtype > 2) return VLA_ERR_DTYPE;
            if (!l.packed || !l.out || (l.out_dtype != VLA_I32 && !l.w_scale)) return VLA_ERR_NULL;
            if (l.N < 128 || l.N % 128 != 0) return VLA_ERR_SHAPE;
            if (!aligned16(l.packed) || !aligned16(l.out) || (reinterpret_cast<uintptr_t>(l.w_scale) & 3u)) return VLA_ERR_ALIGN;
        }
    }
    return VLA_OK;
}

#ifndef VLA_LP_NSCRATCH
#define VLA_LP_NSCRATCH 8
#endif
constexpr int LP_NSCRATCH = VLA_LP_NSCRATCH;      // {int8 [M,K], alpha [M]} scratch sets: the quantiser runs up to seven stages ahead
// Token-tile width of a stage of a large program whose tiles interleave with other stages' tiles: minimise the CTA time of
// the stage, ceil(M / TN) token tiles x cost of a tile's k block.  Measured in steady state on B200 (48 independent stages,
// M = 544, TN = 80..256): a k block costs 0.155 us + 1.25 ns per token with two k blocks per pipeline stage
// (TN <= 160, even K / 128), 0.167 us + 1.25 ns per token with one.
int pick_tn_work(int M, int K) {
    const bool k_even = (K / 128) % 2 == 0;
    int best = 16;
    double best_cost = 1e30;
    for (int tn = 16; tn <= 256; tn += 16) {
        const int tiles_m = (M + tn - 1) / tn;
        if (tn > 16 && (tiles_m * (tn - 16) >= M)) continue;          // a narrower tile covers M with the same count
        const double per_kb = ((tn <= 160 && k_even) ? 0.155 : 0.167) + 1.25e-3 * tn;
        const double cost = tiles_m * per_kb;
        if (cost < best_cost) { best_cost = cost; best = tn; }
    }
    return best;
}

struct LLayout { size_t off_stages, off_counters, off_xq[LP_NSCRATCH], off_xs[LP_NSCRATCH], off_stamps, total; };

LLayout llayout_of(const vla_prog_stage* st, int n) {
    LLayout L{};
    size_t max_xq = 0, max_m = 0;
    for (int s = 0; s < n; ++s) {
        max_xq = std::max(max_xq, (size_t)st[s].M * (size_t)st[s].K);
        max_m = std::max(max_m, (size_t)st[s].M);
    }
    size_t o = round256(sizeof(vla::DevLProg));
    L.off_stages = o;   o += round256(sizeof(vla::LpStage) * (size_t)n);
    L.off_counters = o; o += round256(sizeof(unsigned) * (2 * (size_t)n + 1));
    for (int b = 0; b < LP_NSCRATCH; ++b) { L.off_xq[b] = o; o += round256(max_xq); }
    for (int b = 0; b < LP_NSCRATCH; ++b) { L.off_xs[b] = o; o += round256(4 * max_m); }
#ifdef VLA_LP_STAMPS
    L.off_stamps = o;   o += round256(sizeof(unsigned long long) * 8 * 160 * (size_t)n);
#endif
    L.total = o;
    return L;
}

vla_status check_stages(const vla_prog_stage* st, int n) {
    if (!st) return VLA_ERR_NULL;
    if (n < 1 || n > 4096) return VLA_ERR_SHAPE;
    {                                                         // one kind per program: all stages small, or all large
        const bool large = is_large(st);
        for (int s = 1; s < n; ++s) if ((st[s].M > 16) != large) return VLA_ERR_SHAPE;
        if (large) return check_large(st, n);
    }
    for (int s = 0; s < n; ++s) {
        const vla_prog_stage& a = st[s];
        if (!a.x_bf16 || !a.linears) return VLA_ERR_NULL;
        if (a.M < 1 || a.M > 16 || a.K < 128 || a.K % 128 != 0 || a.K > 8192) return VLA_ERR_SHAPE;
        if (a.n_linears < 1 || a.n_linears > 16) return VLA_ERR_SHAPE;
        if (a.depends != 0 && a.depends != 1) return VLA_ERR_SHAPE;
        if (!aligned16(a.x_bf16) || (a.xq_opt && !aligned16(a.xq_opt)) || (a.x_scale_opt && !aligned16(a.x_scale_opt)))
            return VLA_ERR_ALIGN;
        for (int j = 0; j < a.n_linears; ++j) {
            const vla_prog_linear& l = a.linears[j];
            if (l.out_dtype < 0 || l.out_dtype > 2) return VLA_ERR_DTYPE;
            if (!l.packed || !l.out || (l.out_dtype != VLA_I32 && !l.w_scale)) return VLA_ERR_NULL;
            if (l.N < 128 || l.N % 128 != 0) return VLA_ERR_SHAPE;
            if (!aligned16(l.packed) || !aligned16(l.out) || (reinterpret_cast<uintptr_t>(l.w_scale) & 3u)) return VLA_ERR_ALIGN;
        }
    }
    size_t n_lin = 0;
    for (int s = 0; s < n; ++s) n_lin += (size_t)st[s].n_linears;
    // shared memory of the launch: descriptors + the largest quantised activation matrix + at least two ring slots
    int need = 0;                                             // worst CTA: its stage's activations + two ring slots
    for (int s = 0; s < n; ++s)
        need = std::max(need, ((vla::pg_xq_bytes(st[s].M, st[s].K) + 127) & ~127) + vla::PG_NSLOT_MIN * vla::pg_slot_bytes(st[s].K));
    if ((size_t)vla::pg_off_xq(n, (int)n_lin) + need > (size_t)vla::PG_SMEM_LIMIT) return VLA_ERR_SHAPE;
    return VLA_OK;
}

struct Layout {
    size_t off_stages, off_lins, off_counters, off_stamps, off_act, total;
    int n_lin;
};

Layout layout_of(const vla_prog_stage* st, int n) {
    Layout L{};
    L.n_lin = 0;
    for (int s = 0; s < n; ++s) L.n_lin += st[s].n_linears;
    size_t o = round256(sizeof(DevProg));
    L.off_stages = o;   o += round256(sizeof(DevStage) * (size_t)n);
    L.off_lins = o;     o += round256(sizeof(DevLin) * (size_t)L.n_lin);
    L.off_counters = o; o += round256(sizeof(unsigned) * (2 * (size_t)n + 1));
    L.off_act = o;                                           // cooperative stages: int8 fragments + alpha [16]
    for (int s = 0; s < n; ++s)
        if (!vla::pg_local_quant(st[s].M, st[s].K)) o += round256((size_t)vla::pg_xq_bytes(st[s].M, st[s].K)) + 256;
    L.off_stamps = o;
#ifdef VLA_PROG_STAMPS
    o += round256(sizeof(unsigned long long) * 32 * 256);
#endif
    L.total = o;
    return L;
}


vla_status build_large(const vla_prog_stage* stages, int n_stages, void* prog_dev, size_t prog_bytes, void* stream) {
    using vla::LpStage;
    using vla::DevLProg;
    const LLayout L = llayout_of(stages, n_stages);
    if (prog_bytes < L.total) return VLA_ERR_WORKSPACE;
    int dev = 0, sms = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return VLA_ERR_ARCH;
    }
    if (major != 10 || sms < 1) return VLA_ERR_ARCH;
    uint8_t* base = reinterpret_cast<uint8_t*>(prog_dev);
    std::vector<uint8_t> host(L.off_xq[0] + 64, 0);
    // LpStage is 64-byte aligned (tensor maps): place the table at a 64-byte aligned HOST address with the same offsets
    uint8_t* h = host.data() + ((64 - (reinterpret_cast<uintptr_t>(host.data()) & 63u)) & 63u);
    DevLProg* P = reinterpret_cast<DevLProg*>(h);
    LpStage* S = reinterpret_cast<LpStage*>(h + L.off_stages);
    P->magic = vla::LPROG_MAGIC;
    P->n_stages = n_stages;
    P->qdone = reinterpret_cast<unsigned*>(base + L.off_counters);
    P->gdone = P->qdone + n_stages;
    P->done = P->gdone + n_stages;
    P->stages = reinterpret_cast<const LpStage*>(base + L.off_stages);
#ifdef VLA_LP_STAMPS
    P->stamps = reinterpret_cast<unsigned long long*>(base + L.off_stamps);
    fprintf(stderr, "lprog stamps at offset %zu\n", L.off_stamps);
#else
    P->stamps = nullptr;
#endif
    // Work-minimising token tiles pay as soon as the program has enough tiles to keep every SM busy while stages overlap
    // (measured: the one-step configs[2] program, 297 such tiles, 42.2 -> 38.6 us; a lone (2560,2560) stage, 60 tiles, loses)
    bool long_program = false;
    {
        long long tiles = 0;
        for (int s = 0; s < n_stages; ++s) {
            const vla_prog_stage& a = stages[s];
            int n_total = 0;
            for (int j = 0; j < a.n_linears; ++j) n_total += a.linears[j].N;
            const int tn = pick_tn_work(a.M, a.K);
            tiles += (long long)(n_total / 128) * ((a.M + tn - 1) / tn);
        }
        long_program = 2 * tiles >= 3 * (long long)sms;
    }
    int KS = 2, prev_user[LP_NSCRATCH];
    bool k_even_all = true;
    for (int b = 0; b < LP_NSCRATCH; ++b) prev_user[b] = -1;
    uint32_t x_tile = 0;
    for (int s = 0; s < n_stages; ++s) {
        const vla_prog_stage& a = stages[s];
        LpStage& d = S[s];
        int n_total = 0;
        d.grp.n = a.n_linears;
        d.grp.ct_begin[0] = 0;
        for (int j = 0; j < a.n_linears; ++j) {
            const vla_prog_linear& l = a.linears[j];
            d.grp.packed[j] = reinterpret_cast<const uint8_t*>(l.packed);
            d.grp.beta[j] = l.w_scale;
            d.grp.out[j] = l.out;
            d.grp.N[j] = l.N;
            d.grp.dtype[j] = l.out_dtype;
            d.grp.ct_begin[j + 1] = d.grp.ct_begin[j] + l.N / 128;
            n_total += l.N;
        }
        d.x = reinterpret_cast<const uint4*>(a.x_bf16);
        d.M = a.M;
        d.K = a.K;
        // A stage that can overlap with an independent neighbour (the CTAs it leaves idle start the next stage: tile round
        // robin, `rot`) wants the LEAST TOTAL CTA TIME, not the fewest waves -- if the program is long enough for that to
        // show (`long_program`); a stage that runs alone on the GPU (single stage, dependent chain) and the stages of a short
        // program, whose makespan is one long tile after the quantiser chain, keep gemm_large's wave model.
        const bool overlaps = (s + 1 < n_stages && stages[s + 1].depends == 0) || (s > 0 && a.depends == 0);
        d.TN = (overlaps && long_program) ? pick_tn_work(a.M, a.K) : vla::lg_pick_tn(a.M, n_total, sms, (a.K / 128) % 2 == 0);
        if (vla::lg_pick_ks(d.TN, a.K) != 2) KS = 1;                 // (shared-memory A operand; redone below for ATM)
        if ((a.K / 128) % 2 != 0) k_even_all = false;
        x_tile = std::max(x_tile, ((uint32_t)d.TN * 128u + 1023u) & ~1023u);
        d.tiles_n = n_total / 128;
        d.ntiles = d.tiles_n * ((a.M + d.TN - 1) / d.TN);
        d.x_dep = a.depends > 0 ? 1 : 0;
        const int b = s % LP_NSCRATCH;                        // scratch set of the stage
        d.xq = a.xq_opt ? a.xq_opt : reinterpret_cast<int8_t*>(base + L.off_xq[b]);
        d.xs = a.x_scale_opt ? a.x_scale_opt : reinterpret_cast<float*>(base + L.off_xs[b]);
        d.wait_stage = std::max(a.depends > 0 ? s - a.depends : -1, prev_user[b]);
        prev_user[b] = s;
        d.rot = 0;
        if (vla::lg_encode_x_map(d.tmap, d.xq, a.M, a.K, d.TN) != cudaSuccess) { cudaGetLastError(); return VLA_ERR_CUDA; }
    }
    // The decoded A operand goes to TENSOR MEMORY when every token tile leaves columns for it beside the two accumulators
    // (TN <= 192): a pipeline stage in shared memory then holds X only, and 2-3 times as many X tiles are in flight.
    int max_tn = 0;
    for (int s = 0; s < n_stages; ++s) max_tn = std::max(max_tn, S[s].TN);
#ifdef VLA_LP_NO_ATM
    const bool atm = false;
#else
    const bool atm = max_tn <= 192;
#endif
    // with A in tensor memory a stage costs no shared memory for A, so two k blocks per stage (eight MMAs per barrier round
    // trip of the issuing lane) pay for every token tile: 26.9 -> 23.6 us per prefill step at TN = 192
    if (atm) KS = k_even_all ? 2 : 1;
    const int acc_stride = !atm ? 256 : (max_tn <= 128 ? 128 : 192);
    const int NA = !atm ? 1 : std::min(vla::LP_NA_MAX, (512 - 2 * acc_stride) / (32 * KS));
    const int stride = KS * ((atm ? 0 : vla::LG_A_BYTES) + (int)x_tile);
    // Shared memory: NS {decoded A, X} pipeline stages, NSW packed-weight stages, and the row buffer of the fused quantiser --
    // room for the rows a CTA quantises per stage (at most 16 at a time), in any case for one row.  As many pipeline stages
    // as fit beside the row buffer and a 6-deep weight ring (at least 3, or 2 with two k blocks per stage); one more if a
    // 4-deep weight ring makes room for it.
    const int smem_limit = vla::LG_SMEM_LIMIT - 64;
    auto fixed_bytes = [&](int ns, int nsw) {
        return ns * stride + nsw * KS * vla::LG_W_BYTES + vla::LG_SCALE_BYTES + 1024 + 8 * vla::LG_NBAR + 16 + vla::LP_EXTRA_SMEM;
    };
    int want = 0, one_row = 0;
    for (int s = 0; s < n_stages; ++s) {
        const int rows = std::min(16, (S[s].M + std::min(sms, S[s].M) - 1) / std::min(sms, S[s].M));
        want = std::max(want, 2 * rows * S[s].K * 2);           // two halves: the next chunk's rows load during this chunk's passes
        one_row = std::max(one_row, S[s].K * 2);
    }
    const int ns_floor = atm ? 4 : (KS == 2 ? 2 : 3);
    // the quantiser's chunks: rows per chunk of a stage for a row buffer of `qb` bytes -- double-buffered (a chunk per half, the
    // next chunk's rows load during this chunk's passes) unless that takes more chunks than the whole buffer would: a chunk
    // costs ~1 us of barriers and copy issue whatever its size
    auto chunking = [&](int qb, int K, int rows, int* rpc, int* dbl) {
        const int row_bytes = K * 2, half = (qb / 2) & ~127;
        const int rpc1 = std::max(1, std::min(16, qb / row_bytes)), rpc2 = std::min(16, half / row_bytes);
        const int c1 = (rows + rpc1 - 1) / rpc1, c2 = rpc2 > 0 ? (rows + rpc2 - 1) / rpc2 : (1 << 30);
        *dbl = c2 <= c1 ? 1 : 0;
        *rpc = *dbl ? rpc2 : rpc1;
        return *dbl ? c2 : c1;
    };
    int NS = 0, NSW = vla::LG_SW;
    long long best_chunks = 0;
    // (an EVEN weight ring only: the two decode groups alternate over its stages, and with an odd depth a group would come back
    // to a stage last filled for the OTHER group -- whose copy may not even have landed, so that the parity wait falls through)
    for (int nsw = vla::LG_SW; nsw >= 4; nsw -= 2) {
        int ns = (smem_limit - fixed_bytes(0, nsw) - want) / stride;                  // with the whole row buffer
        if (ns < ns_floor) ns = std::min(ns_floor, (smem_limit - fixed_bytes(0, nsw) - one_row) / stride);   // with a smaller one
        if (ns > vla::LG_NS_MAX) ns = vla::LG_NS_MAX;
        if (ns < NS || ns < 2) continue;
        const int qb = std::min(want, smem_limit - fixed_bytes(ns, nsw)) & ~127;
        long long chunks = 0;                                    // per CTA, over the program
        for (int s = 0; s < n_stages; ++s) {
            int rpc, dbl;
            chunks += chunking(qb, S[s].K, (S[s].M + std::min(sms, S[s].M) - 1) / std::min(sms, S[s].M), &rpc, &dbl);
        }
        // the deepest pipeline first; then a 4-deep weight ring if the row buffer it frees saves chunks
        if (ns > NS || chunks < best_chunks) { NS = ns; NSW = nsw; best_chunks = chunks; }
    }
    if (NS < 2) return VLA_ERR_SHAPE;
    int qbuf = std::min(want, smem_limit - fixed_bytes(NS, NSW));
    qbuf &= ~127;
    if (qbuf < one_row) return VLA_ERR_SHAPE;
    P->KS = KS;
    P->NS = NS;
    P->NSW = NSW;
    P->ATM = atm ? 1 : 0;
    P->acc_stride = acc_stride;
    P->NA = NA;
    P->pad2 = 0;
    P->x_tile = x_tile;
    P->qbuf_bytes = (uint32_t)qbuf;
    P->smem_bytes = fixed_bytes(NS, NSW) + qbuf;
    // with the round robin continued across stages (rot), a stage with fewer tiles than SMs leaves the other CTAs to the next
    // stage: size the grid for the whole program, not for its widest stage
    long long all_tiles = 0;
    for (int s = 0; s < n_stages; ++s) all_tiles += S[s].ntiles;
    int grid = all_tiles < sms ? (int)all_tiles : sms;
    {   // the CTAs wait for each other: all of them must be resident at once
        int per_sm = 0;
        if (vla::lprogram_max_ctas_per_sm(KS, P->ATM, P->smem_bytes, &per_sm) != cudaSuccess) { cudaGetLastError(); return VLA_ERR_CUDA; }
        if (per_sm < 1) return VLA_ERR_CUDA;
        if (grid > per_sm * sms) grid = per_sm * sms;
    }
    for (int s = 0; s < n_stages; ++s) {                       // the quantiser's geometry (lprogram.h)
        S[s].q_rows = S[s].M / grid;
        S[s].q_rem = S[s].M % grid;
        chunking(qbuf, S[s].K, (S[s].M + grid - 1) / grid, &S[s].q_rpc, &S[s].q_dbl);
    }
    {   // Tiles of a stage go to consecutive CTAs starting at `rot` (round robin).  rot is chosen per stage so that the
        // CTAs that get one tile more than the others are the least loaded ones so far (estimated CTA time: k blocks x
        // cost of a k block at the stage's TN); a stage that waits for its predecessor levels the loads.
        std::vector<double> load(grid, 0.0);
        int cont = 0;                                          // where the previous stage's tiles ended
        for (int s = 0; s < n_stages; ++s) {
            if (S[s].wait_stage == s - 1 && s > 0) {
                const double top = *std::max_element(load.begin(), load.end());
                std::fill(load.begin(), load.end(), top);
            }
            const double cost = (S[s].K / 128) * ((KS == 2 ? 0.155 : 0.167) + 1.25e-3 * S[s].TN);
            const int base = S[s].ntiles / grid, rem = S[s].ntiles % grid;
            int best = cont;
            if (rem > 0) {
                double best_max = 1e300, best_sum = 1e300;
                for (int k = 0; k < grid; ++k) {               // candidates in round-robin order: ties keep the continuation
                    const int r = (cont + k) % grid;
                    double mx = 0.0, sum = 0.0;
                    for (int c = 0; c < rem; ++c) { const double v = load[(r + c) % grid]; mx = std::max(mx, v); sum += v; }
                    if (mx < best_max - 1e-9 || (mx < best_max + 1e-9 && sum < best_sum - 1e-9)) { best_max = mx; best_sum = sum; best = r; }
                }
            }
            S[s].rot = best;
            for (int c = 0; c < grid; ++c) load[c] += base * cost;
            for (int c = 0; c < rem; ++c) load[(best + c) % grid] += cost;
            cont = (best + rem) % grid;
        }
    }
    cudaStream_t cs = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(prog_dev, h, L.off_xq[0], cudaMemcpyHostToDevice, cs);
    if (e == cudaSuccess) e = cudaStreamSynchronize(cs);
    if (e != cudaSuccess) { cudaGetLastError(); return VLA_ERR_CUDA; }
#ifdef VLA_LP_STAMPS
    for (int s = 0; s < n_stages && s < 16; ++s)
        fprintf(stderr, "lstage %d: M=%d K=%d TN=%d tiles %d (n %d) wait %d | KS %d NS %d x_tile %u grid %d\n", s, S[s].M, S[s].K,
                S[s].TN, S[s].ntiles, S[s].tiles_n, S[s].wait_stage, KS, NS, x_tile, grid);
#endif
    std::lock_guard<std::mutex> lk(g_mu);
    g_programs[prog_dev] = ProgInfo{grid, n_stages, 0, DevProg{}, true, *P};
    return VLA_OK;
}

}  // namespace

extern "C" {

size_t vla_program_bytes(const vla_prog_stage* stages, int n_stages) {
    if (check_stages(stages, n_stages) != VLA_OK) return 0;
    if (is_large(stages)) return llayout_of(stages, n_stages).total;
    return layout_of(stages, n_stages).total;
}

vla_status vla_program_build(const vla_prog_stage* stages, int n_stages, void* prog_dev, size_t prog_bytes, void* stream) {
    vla_status st = check_stages(stages, n_stages);
    if (st != VLA_OK) return st;
    if (!prog_dev) return VLA_ERR_NULL;
    if (reinterpret_cast<uintptr_t>(prog_dev) & 255u) return VLA_ERR_ALIGN;
    if (is_large(stages)) return build_large(stages, n_stages, prog_dev, prog_bytes, stream);
    const Layout L = layout_of(stages, n_stages);
    if (prog_bytes < L.total) return VLA_ERR_WORKSPACE;
    int dev = 0, sms = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return VLA_ERR_ARCH;
    }
    if (major != 10) return VLA_ERR_ARCH;

    uint8_t* base = reinterpret_cast<uint8_t*>(prog_dev);
    std::vector<uint8_t> host(L.off_act, 0);
    DevProg* P = reinterpret_cast<DevProg*>(host.data());
    DevStage* S = reinterpret_cast<DevStage*>(host.data() + L.off_stages);
    DevLin* Q = reinterpret_cast<DevLin*>(host.data() + L.off_lins);
    P->magic = vla::PROG_MAGIC;
    P->n_stages = n_stages;
    P->n_lin = L.n_lin;
    P->bp = reinterpret_cast<unsigned*>(base + L.off_counters);
    P->cnt = P->bp + n_stages;
    P->done = P->cnt + n_stages;
#ifdef VLA_PROG_STAMPS
    P->stamps = reinterpret_cast<unsigned long long*>(base + L.off_stamps);
#else
    P->stamps = nullptr;
#endif
    P->stages = reinterpret_cast<const DevStage*>(base + L.off_stages);
    P->lins = reinterpret_cast<const DevLin*>(base + L.off_lins);
    int li = 0, max_m = 0, phase = 0, max_phase_gran = 0, phase_gran = 0, max_need = 0, n_coop = 0;
    size_t act = L.off_act;
    for (int s = 0; s < n_stages; ++s) {
        const vla_prog_stage& a = stages[s];
        DevStage& d = S[s];
        d.x = reinterpret_cast<const uint4*>(a.x_bf16);
        d.xq_out = a.xq_opt;
        d.xs_out = a.x_scale_opt;
        d.coop = nullptr;
        if (!vla::pg_local_quant(a.M, a.K)) {
            d.coop = base + act;
            act += round256((size_t)vla::pg_xq_bytes(a.M, a.K)) + 256;
            ++n_coop;
        }
        max_need = std::max(max_need, ((vla::pg_xq_bytes(a.M, a.K) + 127) & ~127) + vla::PG_NSLOT_MAX * vla::pg_slot_bytes(a.K));
        d.inv_cpr = (uint32_t)((0x100000000ull + (unsigned)(a.K / 16) - 1u) / (unsigned)(a.K / 16));
        d.M = (int16_t)a.M;
        d.K = (int16_t)a.K;
        d.flags = (int16_t)((s == 0) ? 0 : a.depends);      // nothing precedes the first stage
        if (d.flags & 1) { ++phase; phase_gran = 0; }        // a dependent stage opens a new phase
        d.phase = phase;
        if (a.M > max_m) max_m = a.M;
        d.lin_begin = li;
        d.n_lin = (int16_t)a.n_linears;
        int gran = 0;
        for (int j = 0; j < a.n_linears; ++j, ++li) {
            const vla_prog_linear& l = a.linears[j];
            Q[li].packed = reinterpret_cast<const uint8_t*>(l.packed);
            Q[li].beta = l.w_scale;
            Q[li].out = l.out;
            Q[li].N = l.N;
            Q[li].dtype = l.out_dtype;
            Q[li].gran_begin = gran;
            Q[li].pad = 0;
            gran += l.N / 32;
        }
        d.granules = gran;
        phase_gran += gran;
        if (phase_gran > max_phase_gran) max_phase_gran = phase_gran;
    }
    P->n_phases = phase + 1;
    int grid = max_phase_gran < sms ? max_phase_gran : sms;
    // dynamic shared memory: everything up to the activation region, the largest activation matrix, and as many ring
    // slots as fit (a CTA whose own stages need less activation room gets more slots)
    const int fixed = vla::pg_off_xq(n_stages, L.n_lin);
    int smem = fixed + max_need;
    if (smem > vla::PG_SMEM_LIMIT) smem = vla::PG_SMEM_LIMIT;
    P->smem_bytes = smem;
    P->gate = VLA_PROG_GATE;
    P->n_coop = n_coop;
    P->pad = 0;
    if (P->n_phases > 1 || n_coop > 0) {
        // CTAs of a multi-phase program wait for each other: all of them must be resident at once
        int per_sm = 0;
        if (vla::program_max_ctas_per_sm(max_m, smem, &per_sm) != cudaSuccess) { cudaGetLastError(); return VLA_ERR_CUDA; }
        if (per_sm < 1) return VLA_ERR_CUDA;
        if (grid > per_sm * sms) grid = per_sm * sms;
    }
    // Split the grid among the stages of each phase so that the slowest group finishes as early as possible.  Model of a
    // stage on c CTAs, in SM cycles, from per-CTA clock stamps on B200:
    //     t(c) = start + ceil(granules / c) * g                                   (KB = K / 128, 1 KiB pieces per granule)
    //     15-way k split:  M <= 8:  g = F1A + F1B KB        M > 8:  g = F2A + F2B KB
    //     team mode     :  M <= 8:  g = T1A + T1B KB        M > 8:  g = T2A + T2B KB      (prog_team_mode(), program.h)
    //     start = START0 + START1 * (16-element tasks) for a locally quantised stage, START_COOP for a cooperative one
    auto start_cycles = [&](int s) {                          // fused quant before the first granule (measured, profiles/r02*)
        return vla::pg_local_quant(S[s].M, S[s].K) ? VLA_PG_START0 + VLA_PG_START1 * (S[s].M * (S[s].K / 16)) : VLA_PG_START_COOP;
    };
    auto stage_time = [&](int s, int c) {
        const double KB = S[s].K / 128;
        const bool team = vla::prog_team_mode(S[s].granules, c);
        const double g = team ? (S[s].M > 8 ? VLA_PG_T2A + VLA_PG_T2B * KB : VLA_PG_T1A + VLA_PG_T1B * KB)
                              : (S[s].M > 8 ? VLA_PG_F2A + VLA_PG_F2B * KB : VLA_PG_F1A + VLA_PG_F1B * KB);
        return start_cycles(s) + (double)((S[s].granules + c - 1) / c) * g;
    };
    for (int s0 = 0; s0 < n_stages;) {
        int s1 = s0 + 1;
        while (s1 < n_stages && S[s1].phase == S[s0].phase) ++s1;
        const int ns = s1 - s0;
        if (ns > grid) return VLA_ERR_SHAPE;                 // more independent stages in one phase than CTAs
        // smallest finish time T for which the groups fit in the grid; candidates: t(c) of every stage and group size
        std::vector<double> cand;
        for (int s = s0; s < s1; ++s)
            for (int c = 1; c <= grid && c <= S[s].granules; ++c) cand.push_back(stage_time(s, c));
        std::sort(cand.begin(), cand.end());
        auto fewest = [&](int s, double T) {                  // smallest group that finishes stage s by T (or -1);
            const int cmax = S[s].granules < grid ? S[s].granules : grid;      // t(c) is not monotone at the team threshold
            for (int c = 1; c <= cmax; ++c)
                if (stage_time(s, c) <= T + 1e-9) return c;
            return -1;
        };
        auto need = [&](double T) {
            int sum = 0;
            for (int s = s0; s < s1; ++s) {
                const int c = fewest(s, T);
                if (c < 0) return -1;
                sum += c;
            }
            return sum;
        };
        size_t lo = 0, hi = cand.size() - 1;
        {                                                     // feasibility is monotone in T; the largest candidate may still
            const int n = need(cand[hi]);                     // need more than `grid` CTAs only if ns > grid (excluded above)
            if (n < 0 || n > grid) lo = hi;
        }
        while (lo < hi) {
            const size_t mid = (lo + hi) / 2;
            const int n = need(cand[mid]);
            if (n >= 0 && n <= grid) hi = mid; else lo = mid + 1;
        }
        int given = 0;
        for (int s = s0; s < s1; ++s) {
            int c = fewest(s, cand[lo]);
            if (c < 1) c = 1;
            S[s].cta_count = c;
            given += c;
        }
        while (given > grid) {                               // (only if the model was infeasible) shrink the largest group
            int big = s0;
            for (int s = s0; s < s1; ++s) if (S[s].cta_count > S[big].cta_count) big = s;
            --S[big].cta_count;
            --given;
        }
        while (given < grid) {                               // spare CTAs: to the group that finishes last, if one more helps
            int best = -1;
            for (int s = s0; s < s1; ++s)
                if (S[s].cta_count < S[s].granules && stage_time(s, S[s].cta_count + 1) <= stage_time(s, S[s].cta_count) &&
                    (best < 0 || stage_time(s, S[s].cta_count) > stage_time(best, S[best].cta_count))) best = s;
            if (best < 0) {                                   // nobody gains: park the spare CTAs on the largest group
                best = s0;
                for (int s = s0; s < s1; ++s) if (S[s].granules > S[best].granules) best = s;
            }
            ++S[best].cta_count;
            ++given;
        }
        int begin = 0;
        for (int s = s0; s < s1; ++s) { S[s].cta_begin = begin; begin += S[s].cta_count; }
        if (s1 < n_stages) S[s1 - 1].flags |= 2;             // publish: the next phase opens with a dependent stage
        s0 = s1;
    }

#ifdef VLA_PROG_STAMPS
    for (int s = 0; s < n_stages && s < 16; ++s)
        fprintf(stderr, "stage %d: M=%d K=%d granules=%d phase=%d ctas [%d,+%d) model %.0f cycles\n", s, S[s].M, S[s].K,
                S[s].granules, S[s].phase, S[s].cta_begin, S[s].cta_count, stage_time(s, S[s].cta_count));
#endif
    cudaStream_t cs = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(prog_dev, host.data(), host.size(), cudaMemcpyHostToDevice, cs);
    // the scratch of cooperative stages starts at zero: the fragments of padding rows (M .. 8 or 16) are never written
    if (e == cudaSuccess && L.total > L.off_act) e = cudaMemsetAsync(base + L.off_act, 0, L.total - L.off_act, cs);
    if (e == cudaSuccess) e = cudaStreamSynchronize(cs);
    if (e != cudaSuccess) { cudaGetLastError(); return VLA_ERR_CUDA; }
    std::lock_guard<std::mutex> lk(g_mu);
    g_programs[prog_dev] = ProgInfo{grid, n_stages, max_m, *P, false, vla::DevLProg{}};
    return VLA_OK;
}

vla_status vla_program_run(const void* prog_dev, void* stream) {
    if (!prog_dev) return VLA_ERR_NULL;
    ProgInfo info;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        auto it = g_programs.find(prog_dev);
        if (it == g_programs.end()) return VLA_ERR_VALUE;
        info = it->second;
    }
    cudaError_t e = info.large ? vla::launch_lprogram(info.lheader, info.grid, (cudaStream_t)stream)
                               : vla::launch_program(info.header, info.grid, info.max_m, (cudaStream_t)stream);
    if (e != cudaSuccess) { cudaGetLastError(); return VLA_ERR_CUDA; }
    return VLA_OK;
}

vla_status vla_program_run_host_async(const void* prog_dev, const vla_copy* in, int n_in, const vla_copy* out, int n_out,
                                      void* stream) {
    if (!prog_dev || (n_in > 0 && !in) || (n_out > 0 && !out)) return VLA_ERR_NULL;
    if (n_in < 0 || n_out < 0) return VLA_ERR_SHAPE;
    for (int i = 0; i < n_in; ++i) if (!in[i].host || !in[i].dev) return VLA_ERR_NULL;
    for (int i = 0; i < n_out; ++i) if (!out[i].host || !out[i].dev) return VLA_ERR_NULL;
    cudaStream_t cs = (cudaStream_t)stream;
    for (int i = 0; i < n_in; ++i)
        if (cudaMemcpyAsync(in[i].dev, in[i].host, in[i].bytes, cudaMemcpyHostToDevice, cs) != cudaSuccess) {
            cudaGetLastError();
            return VLA_ERR_CUDA;
        }
    vla_status st = vla_program_run(prog_dev, stream);
    if (st != VLA_OK) return st;
    for (int i = 0; i < n_out; ++i)
        if (cudaMemcpyAsync(out[i].host, out[i].dev, out[i].bytes, cudaMemcpyDeviceToHost, cs) != cudaSuccess) {
            cudaGetLastError();
            return VLA_ERR_CUDA;
        }
    return VLA_OK;
}

vla_status vla_program_run_host(const void* prog_dev, const vla_copy* in, int n_in, const vla_copy* out, int n_out,
                                void* stream) {
    vla_status st = vla_program_run_host_async(prog_dev, in, n_in, out, n_out, stream);
    if (st != VLA_OK) return st;
    if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) { cudaGetLastError(); return VLA_ERR_CUDA; }
    return VLA_OK;
}

vla_status vla_ternary_gemm_grouped(const vla_prog_linear* lins, int n_linears, const int8_t* xq, const float* x_scale,
                                    int M, int K, vla_path path, void* stream) {
    if (!lins || !xq) return VLA_ERR_NULL;
    if (n_linears < 1 || n_linears > 8 || M < 1 || K < 128 || K % 128 != 0 || K > 65536) return VLA_ERR_SHAPE;
    if ((int)path < 0 || (int)path > 3) return VLA_ERR_DTYPE;
    if (!aligned16(xq) || (x_scale && !aligned16(x_scale))) return VLA_ERR_ALIGN;
    bool need_scale = false;
    for (int j = 0; j < n_linears; ++j) {
        const vla_prog_linear& l = lins[j];
        if (l.out_dtype < 0 || l.out_dtype > 2) return VLA_ERR_DTYPE;
        if (!l.packed || !l.out || (l.out_dtype != VLA_I32 && !l.w_scale)) return VLA_ERR_NULL;
        if (l.N < 128 || l.N % 128 != 0) return VLA_ERR_SHAPE;
        if (!aligned16(l.packed) || !aligned16(l.out) || (reinterpret_cast<uintptr_t>(l.w_scale) & 3u)) return VLA_ERR_ALIGN;
        need_scale = need_scale || l.out_dtype != VLA_I32;
    }
    if (need_scale && !x_scale) return VLA_ERR_NULL;
    int n_total = 0;                                        // the grouped launch runs the group as one [sum N, K] linear
    for (int j = 0; j < n_linears; ++j) n_total += lins[j].N;
    const bool large = (path == VLA_PATH_LARGE) || (path == VLA_PATH_AUTO && vla_ternary_auto_path(M, n_total, K) == VLA_PATH_LARGE);
    if (!large) {                                           // small-M: one launch per linear (or use a program)
        for (int j = 0; j < n_linears; ++j) {
            vla_status st = vla_ternary_gemm(lins[j].packed, lins[j].w_scale, xq, x_scale, M, lins[j].N, K, lins[j].out,
                                             (vla_dtype)lins[j].out_dtype, path, nullptr, 0, stream);
            if (st != VLA_OK) return st;
        }
        return VLA_OK;
    }
    int dev = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        cudaGetLastError();
        return VLA_ERR_ARCH;
    }
    if (major != 10) return VLA_ERR_ARCH;
    vla::LgGroup g = {};
    g.n = n_linears;
    g.ct_begin[0] = 0;
    for (int j = 0; j < n_linears; ++j) {
        g.packed[j] = reinterpret_cast<const uint8_t*>(lins[j].packed);
        g.beta[j] = lins[j].w_scale;
        g.out[j] = lins[j].out;
        g.N[j] = lins[j].N;
        g.dtype[j] = lins[j].out_dtype;
        g.ct_begin[j + 1] = g.ct_begin[j] + lins[j].N / 128;
    }
    cudaError_t e = vla::launch_gemm_large_grouped(g, xq, x_scale, M, K, (cudaStream_t)stream);
    if (e != cudaSuccess) { cudaGetLastError(); return VLA_ERR_CUDA; }
    return VLA_OK;
}

vla_status vla_program_release(const void* prog_dev) {
    if (!prog_dev) return VLA_ERR_NULL;
    std::lock_guard<std::mutex> lk(g_mu);
    return g_programs.erase(prog_dev) ? VLA_OK : VLA_ERR_VALUE;
}

}  // extern "C"
