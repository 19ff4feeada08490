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
    uint2* xq;                 // int8 [M,K]   (inside the program buffer unless the caller asked for it)
    float* xs;                 // fp32 [M]
    int16_t M;
    int16_t n_lin;
    int16_t flags;             // bit 0 "depends": x is written by earlier phases of this program
                               // bit 1 "publish": last stage of its phase AND the next phase depends -> count in bp
                               // bit 2 "rows in group": the stage's own CTA group quantises its rows (else the whole grid)
    int16_t K;
    int lin_begin;
    int granules;              // sum over its linears of N/32
    int phase;                 // stages of one phase are independent and run concurrently on disjoint CTA groups
    int cta_begin, cta_count;  // the CTA group of this stage: [cta_begin, cta_begin + cta_count)
    int row_begin;             // (running sum of M over all earlier stages) % grid: row r is quantised by CTA (row_begin + r) % grid
};

struct DevProg {
    uint32_t magic;
    int n_stages;
    int n_lin;
    int n_phases;
    unsigned* bp;              // [n_phases] CTAs that finished phase p             (target gridDim.x)
    unsigned* b2;              // [n_stages] rows of stage s that are quantised      (target M_s)
    unsigned* done;            // [1]        CTAs that finished the program; the last one re-zeroes the counters
    const DevStage* stages;
    const DevLin* lins;
};

// Team mode of the program kernel (gemm_program.cu): the stage's group runs three 5-warp teams on three granules at
// once.  Needs K <= 2880 (a five-way k split whose B fragments still fit in 9 x uint4 per thread) and at least two
// granules per team and CTA.  One definition for the kernel and for the partition model of the program compiler.
#if defined(__CUDACC__)
__host__ __device__
#endif
inline bool prog_team_mode(int K, int granules, int cta_count) { return K / 64 <= 45 && granules >= 6 * cta_count; }

}  // namespace vla
