// pack.cu -- weight packer / unpacker (offline, once per tensor).
// One thread per 32-bit packed word = 16 consecutive k of one output channel.  Layout: common.cuh.
#include "common.cuh"
#include "kernels.h"

namespace vla {

// word index -> (n, k0)
__device__ __forceinline__ void word_coords(size_t word, int K, int& n, int& k0) {
    int j = (int)(word & 3);
    int lane = (int)((word >> 2) & 31);
    size_t blk = word >> 7;                         // 512-byte block index = n32 * (K/64) + k64
    int blocks_k = K / BLK_K;
    int n32 = (int)(blk / blocks_k), k64 = (int)(blk % blocks_k);
    int g = lane >> 2, t = lane & 3;
    n = n32 * BLK_N + j * 8 + g;
    k0 = k64 * BLK_K + t * 16;
}

__global__ void pack_kernel(const int8_t* __restrict__ w, int N, int K, uint32_t* __restrict__ packed, int* __restrict__ bad) {
    size_t word = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t nwords = (size_t)N * K / 16;
    if (word >= nwords) return;
    int n, k0;
    word_coords(word, K, n, k0);
    uint4 v = *reinterpret_cast<const uint4*>(w + (size_t)n * K + k0);
    uint32_t r[4] = {v.x, v.y, v.z, v.w};
    uint32_t out = 0;
    bool ok = true;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            int q = (int)(int8_t)((r[i] >> (8 * b)) & 0xFF);
            ok = ok && (q >= -1) && (q <= 1);
            out |= ((uint32_t)q & 3u) << (8 * b + 2 * i);
        }
    packed[word] = out;
    if (!ok) atomicOr(bad, 1);
}

__global__ void unpack_kernel(const uint32_t* __restrict__ packed, int N, int K, int8_t* __restrict__ w) {
    size_t word = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t nwords = (size_t)N * K / 16;
    if (word >= nwords) return;
    int n, k0;
    word_coords(word, K, n, k0);
    uint32_t p = packed[word];
    uint32_t r[4] = {0, 0, 0, 0};
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            int c = (p >> (8 * b + 2 * i)) & 3;
            int q = (c ^ 2) - 2;                     // sign-extend the 2-bit two's-complement code
            r[i] |= ((uint32_t)q & 0xFFu) << (8 * b);
        }
    *reinterpret_cast<uint4*>(w + (size_t)n * K + k0) = make_uint4(r[0], r[1], r[2], r[3]);
}

cudaError_t launch_pack(const int8_t* w, int N, int K, void* packed, int* bad_flag, cudaStream_t s) {
    size_t nwords = (size_t)N * K / 16;
    count_launch();
    pack_kernel<<<(unsigned)((nwords + 255) / 256), 256, 0, s>>>(w, N, K, (uint32_t*)packed, bad_flag);
    return cudaGetLastError();
}

cudaError_t launch_unpack(const void* packed, int N, int K, int8_t* w, cudaStream_t s) {
    size_t nwords = (size_t)N * K / 16;
    count_launch();
    unpack_kernel<<<(unsigned)((nwords + 255) / 256), 256, 0, s>>>((const uint32_t*)packed, N, K, w);
    return cudaGetLastError();
}

}  // namespace vla
