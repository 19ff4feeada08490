// gemm_large.cuh -- tile constants and small helpers shared by the tcgen05 kernels (gemm_large.cu: one launch per
// linear / group; gemm_lprog.cu: the persistent multi-stage form with fused activation quant).
#pragma once
#include <cstdint>
#include "common.cuh"

namespace vla {

constexpr int LG_THREADS = 15 * 32;
constexpr int LG_SW = 6;                                // most packed-weight stages (4 KiB per k block each)
constexpr int LG_SMEM_LIMIT = 232448;                   // dynamic shared memory a CTA may opt in to (227 KB)
constexpr int LG_NS_MAX = 8;                            // {decoded A, X} stages
constexpr int LG_A_BYTES = TILE_N * TILE_K;             // 16384 decoded int8
constexpr int LG_W_BYTES = TILE_BYTES;                  // 4096 packed
constexpr int LG_SCALE_BYTES = 4 * 256 * 4;             // per epilogue warp: alpha_m * beta of the tile's tokens
constexpr int LG_NBAR = 2 * LG_SW + 2 * LG_NS_MAX + 4;

__host__ __device__ inline uint32_t lg_stage_stride(int TN) { return LG_A_BYTES + (((uint32_t)TN * TILE_K + 1023u) & ~1023u); }

__device__ __forceinline__ uint4 lds128_nv(uint32_t addr) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
    return r;
}

// Cursor over a ring of `n` slots walked once per pipeline iteration: slot, phase parity of the slot's CURRENT use, and whether
// the ring has wrapped (= the slot has been used before).  Kept incrementally: `it % n` and `it / n` with a run-time n cost
// ~50 dependent instructions per iteration in the single-thread roles (the MMA-issuing lane, the producers).
struct RingCur {
    uint32_t s = 0, ph = 0;
    bool wrapped = false;
    __device__ __forceinline__ void next(uint32_t n) { if (++s == n) { s = 0; ph ^= 1u; wrapped = true; } }
};

// Token-tile width TN (multiple of 16, <= 256) for a persistent grid of `sms` CTAs (gemm_large.cu)
int lg_pick_tn(int M, int N, int sms, bool k_even);
// tensor map (128 bytes, 64-byte aligned) of the int8 activations xq [M,K] for token tiles of TN
cudaError_t lg_encode_x_map(void* tmap_out, const int8_t* xq, int M, int K, int TN);
// k blocks per pipeline stage for a token tile of TN
inline int lg_pick_ks(int TN, int K) { return (TN <= 160 && (K / TILE_K) % 2 == 0) ? 2 : 1; }

}  // namespace vla
