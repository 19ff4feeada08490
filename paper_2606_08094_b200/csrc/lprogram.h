// lprogram.h -- device-side form of a LARGE program: stages with M > 16 tokens, executed by ONE persistent tcgen05
// kernel (gemm_lprog.cu).  A stage is Eq. 4 end to end: the CTAs quantise the rows of x
// cooperatively into an int8 scratch (row r by CTA r mod grid), meet on a grid-wide counter, and then walk the stage's
// 128-channel x TN-token tiles exactly as gemm_large_kernel does.  Stages run in order; a stage with depends = 1 starts
// its quantisation only after every CTA has stored its tiles of the previous stage.
#pragma once
#include <cstdint>
#include "kernels.h"

namespace vla {

constexpr uint32_t LPROG_MAGIC = 0x564C414Cu;   // "VLAL"
constexpr int LP_NA_MAX = 8;          // most A stages of the ATM form (decoded weights in tensor memory)
constexpr int LP_EXTRA_SMEM = 512 + 16 * LP_NA_MAX;   // behind gemm_large's layout: quantiser row absmax [16], scales float4 [16], its mbarrier, and the
                                     // alignment slack of its row buffer (DevLProg::qbuf_bytes more bytes follow)

struct alignas(64) LpStage {
    unsigned char tmap[128];   // CUtensorMap of xq [M,K] int8: box [128 k, TN tokens], SWIZZLE_128B
    LgGroup grp;               // the linears that consume x (per-output-group scales), as one [sum N, K] tile walk
    const uint4* x;            // bf16 [M,K]
    int8_t* xq;                // int8 [M,K]: the caller's xq_opt, else one of the program's scratch sets
    float* xs;                 // alpha [M]: the caller's x_scale_opt, else scratch
    int M, K, TN;
    int wait_stage;            // quantisation of this stage starts after gdone[wait_stage] == grid (-1: at once):
                               // the previous stage if depends = 1, and the last stage that used the same scratch
    int tiles_n, ntiles;       // channel tiles of the group, tiles of the stage
    int rot;                   // tile t runs on CTA (t + rot) mod grid
    // the fused quantiser's geometry, fixed by the host once the grid is known (no division in the kernel):
    int q_rows, q_rem;         // CTA b quantises M / grid rows, + 1 if b < M mod grid (rows b, b + grid, ...)
    int q_rpc;                 // rows per chunk of the row buffer (<= 16)
    int q_dbl;                 // 1: a chunk fits HALF the row buffer -> the next chunk's copies fly during this chunk's passes
    int x_dep;                 // 1: x is written inside this launch (depends > 0): proxy fence before the bulk copies
};

struct DevLProg {
    uint32_t magic;
    int n_stages;
    int KS;                    // k blocks (of 128) per pipeline stage, one value for the whole program
    int NS;                    // {decoded A, X} pipeline stages
    uint32_t x_tile;           // bytes reserved per X tile (the widest token tile of the program, 1 KiB aligned)
    int smem_bytes;
    uint32_t qbuf_bytes;       // row buffer of the quantiser (shared memory); two halves of qbuf_bytes / 2 (128-byte aligned) when double-buffered
    int NSW;                   // packed-weight stages in use (<= LG_SW)
    int ATM;                   // 1: decoded A operand in tensor memory (every token tile <= 192), pipeline stages hold X only
    int acc_stride;            // ATM: TMEM columns per accumulator (128 or 192); the A ring starts at column 2 * acc_stride
    int NA;                    // ATM: A stages of KS x 32 columns
    int pad2;
    unsigned* qdone;           // [n_stages] CTAs that have quantised their rows of stage s      (target gridDim.x)
    unsigned* gdone;           // [n_stages] CTAs that have stored their tiles of stage s         (target gridDim.x)
    unsigned* done;            // [1]        CTAs past their last counter access; the last one re-zeroes the counters
    const LpStage* stages;
    unsigned long long* stamps; // debug builds only (VLA_LP_STAMPS): [n_stages][grid][8] globaltimer stamps
};

cudaError_t launch_lprogram(const DevLProg& prog, int grid, cudaStream_t s);
cudaError_t lprogram_max_ctas_per_sm(int KS, int atm, int smem_bytes, int* out);

}  // namespace vla
