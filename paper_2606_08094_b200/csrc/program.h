// program.h -- device-side form of a compiled "program" of ternary linears (internal to libvlaternary.so).
// A program is a list of STAGES; a stage is one bf16 activation matrix x [M,K] (M <= 16) and the
// ternary linears that consume it (q|k|v share one input, gate|up share one input: the per-output-group
// scales beta_g(n) of Eq. 4).  A stage with depends = 1 opens a new PHASE and may read what earlier
// phases wrote; the stages of one phase are independent of each other.
#pragma once
#include <cstdint>

namespace vla {

constexpr uint32_t PROG_MAGIC = 0x564C4150u;   // "VLAP"

struct DevLin {
    const uint8_t* packed;     // packed W [N,K]
    const float* beta;         // one fp32
    void* out;                 // [M,N]
    int N;
    int dtype;                 // vla_dtype
    int gran_begin;            // first 32-channel granule of this linear within its stage
    int pad;
};

struct DevStage {
    const uint4* x;            // bf16 [M,K]
    int8_t* xq_out;            // optional: int8 [M,K] the caller asked for (else null)
    float* xs_out;             // optional: alpha [M] the caller asked for (else null)
    uint8_t* coop;             // cooperative quant: scratch in the program buffer, [pg_xq_bytes] int8 fragments then
                               // alpha [16]; null: the stage is small and every CTA of its group quantises it locally
    int16_t M;
    int16_t n_lin;
    int16_t flags;             // bit 0 "depends": x is written by earlier phases of this program
                               // bit 1 "publish": last stage of its phase AND the next phase depends -> count in bp
    int16_t K;
    int lin_begin;
    int granules;              // sum over its linears of N/32
    int phase;                 // stages of one phase are independent and run concurrently on disjoint CTA groups
    int cta_begin, cta_count;  // the CTA group of this stage: [cta_begin, cta_begin + cta_count)
    uint32_t inv_cpr;          // ceil(2^32 / (K/16)): f / (K/16) == umulhi(f, inv_cpr) for the quantiser's task index f
};

struct DevProg {
    uint32_t magic;
    int n_stages;
    int n_lin;
    int n_phases;
    int smem_bytes;            // dynamic shared memory of the launch (after alignment): ring slots fill what the
                               // descriptors and this CTA's quantised activations leave free
    int gate;                  // 1: the weight ring waits (after its first chunk) until this CTA's first activations landed
    int n_coop;                // stages with cooperative quant
    int pad;
    unsigned* bp;              // [n_stages] bp[p] = CTAs that finished phase p     (target gridDim.x)
    unsigned* cnt;             // [n_stages] cnt[s] = rows of cooperative stage s that are quantised (target M_s)
    unsigned* done;            // [1]        CTAs past their last counter access; the last one re-zeroes the counters
    unsigned long long* stamps;// debug builds only (VLA_PROG_STAMPS): per-CTA clock stamps inside the program buffer
    const DevStage* stages;
    const DevLin* lins;
};

#ifndef VLA_PG_SLOT_PIECES
#define VLA_PG_SLOT_PIECES 30
#endif
// ---- shared-memory map of program_kernel (one definition for the kernel and the host-side sizing)
constexpr int PG_SLOT_PIECES = VLA_PG_SLOT_PIECES;                    // most 1 KiB pieces (32 channels x 128 k) per ring chunk
constexpr int PG_NSLOT_MAX = 12;
constexpr int PG_NSLOT_MIN = 2;
#ifndef VLA_PG_TEAMS
#define VLA_PG_TEAMS 3
#endif
#ifndef VLA_PG_QNB
#define VLA_PG_QNB 3
#endif
constexpr int PG_TEAMS = VLA_PG_TEAMS, PG_TW = 5;     // teams of five consumer warps
constexpr int PG_W = PG_TEAMS * PG_TW;                // consumer warps (+ 1 producer warp)
constexpr int PG_QNB = VLA_PG_QNB;                    // 16-element quant tasks a thread holds per round
constexpr int PG_RED_STRIDE = 36;                     // ints per token row of an accumulation tile (bank-conflict free)
constexpr int PG_RED_BUF_INTS = 16 * PG_RED_STRIDE;   // one [16 tokens][32 channels] int32 tile
constexpr int PG_RED_INTS = 2 * PG_TEAMS * PG_RED_BUF_INTS;
constexpr int PG_OFF_BAR = 0;                         // full[12] | empty[12] | go | xq (fragments pulled)
constexpr int PG_OFF_ALPHA = 208;                     // float4[16]: alpha_m, 1/alpha_m * (1 -+ 2^-19), -
constexpr int PG_OFF_BETA = 464;                      // float[16]
constexpr int PG_OFF_ROWMAX = 528;                    // unsigned[16]
constexpr int PG_OFF_MISC = 592;                      // unsigned[4]
constexpr int PG_OFF_GOT = 608;                       // unsigned[12]: newest chunk seen to have landed, per ring slot
constexpr int PG_OFF_RED = 704;
constexpr int PG_OFF_INFO = PG_OFF_RED + PG_RED_INTS * 4;
constexpr int PG_SMEM_LIMIT = 232448 - 128;           // 227 KB minus the alignment slack

#if defined(__CUDACC__)
#define VLA_HD __host__ __device__
#else
#define VLA_HD
#endif
VLA_HD inline int pg_round(int b, int a) { return (b + a - 1) / a * a; }
// bytes before the quantised-activation region: barriers, scales, tiles, stage digest, descriptor tables
VLA_HD inline int pg_off_desc(int n_stages) { return PG_OFF_INFO + pg_round(4 * n_stages, 16); }
VLA_HD inline int pg_off_xq(int n_stages, int n_lin) {
    return pg_round(pg_off_desc(n_stages) + n_stages * (int)sizeof(DevStage) + n_lin * (int)sizeof(DevLin), 128);
}
// int8 activations of a stage as mma B fragments: [K/64][token tiles][32 lanes][16 B]
VLA_HD inline int pg_xq_bytes(int M, int K) { return (M > 8 ? 16 : 8) * K; }
// a stage this small (in 16-element tasks) is quantised by every CTA of its group for itself
VLA_HD inline bool pg_local_quant(int M, int K) { return M * (K / 16) <= PG_QNB * PG_W * 32; }
// ring chunks of a granule (K/128 pieces): as few as fit a slot, of equal size
VLA_HD inline int pg_chunks(int KB) { return (KB + PG_SLOT_PIECES - 1) / PG_SLOT_PIECES; }
VLA_HD inline int pg_chunk_pieces(int KB) { const int n = pg_chunks(KB); return (KB + n - 1) / n; }
// the ring slot of a CTA holds the largest chunk of the stages it works on
VLA_HD inline int pg_slot_bytes(int K) { return pg_chunk_pieces(K / 128) * 1024; }

// Team mode of the program kernel (gemm_program.cu): the stage's group runs three 5-warp teams on three granules at
// once; needs at least one granule per team and CTA.  Otherwise all 15 consumer warps split the k blocks of one granule.
// One definition for the kernel and for the partition model of the program compiler.
VLA_HD inline bool prog_team_mode(int granules, int cta_count) { return granules >= PG_TEAMS * cta_count; }

}  // namespace vla
