#include <cstdio>
#include "../csrc/common.cuh"
using namespace vla;
// mode bit0: commit per group of 4 MMAs; bit1: a try_wait on a completed barrier per group; bit2: tcgen05 fence per group
__global__ void __launch_bounds__(64, 1) probe(int groups, int n, int mode) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* base_ptr = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t sA = base, sB = base + 4 * 16384, sBar = sB + 4 * 32768;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < (4 * 16384 + 4 * 32768) / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(base_ptr)[i] = 0x01010101u;
    fence_proxy_async_smem();
    if (threadIdx.x == 0) { for (int b = 0; b < 8; ++b) mbar_init(sBar + 8 * b, 1); fence_barrier_init(); }
    if (warp == 1) tmem_alloc(sBar + 64, 256);
    tc_fence_before(); __syncthreads(); tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(base_ptr + 4 * 16384 + 4 * 32768 + 64);
    if (warp == 0 && lane == 0) {
        mbar_arrive(sBar + 8 * 7);          // barrier 7: phase 0 complete forever
        const uint32_t idesc = umma_idesc_i8(128, n);
        for (int g = 0; g < groups; ++g) {
            const int st = g & 3;
            if (mode & 2) mbar_wait(sBar + 8 * 7, 0);
            if (mode & 4) tc_fence_after();
            const uint64_t a = umma_desc_k_sw128(sA + st * 16384), b = umma_desc_k_sw128(sB + st * 32768);
#pragma unroll
            for (int k = 0; k < 4; ++k) mma_i8_ss(tmem_base, a + 2 * k, b + 2 * k, idesc, (g | k) != 0);
            if (mode & 1) mma_commit(sBar + 8 * (g & 3) );
        }
        mma_commit(sBar + 8 * 4); mbar_wait(sBar + 8 * 4, 0);
    }
    tc_fence_before(); __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, 256);
}
int main() {
    const int smem = 4 * 16384 + 4 * 32768 + 1024 + 128;
    cudaFuncSetAttribute(probe, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    const int groups = 5000;
    for (int n : {96, 256})
    for (int mode : {0, 1, 2, 4, 3, 7}) {
        probe<<<148, 64, smem>>>(groups, n, mode);
        cudaEventRecord(a); probe<<<148, 64, smem>>>(groups, n, mode); cudaEventRecord(b); cudaDeviceSynchronize();
        float ms; cudaEventElapsedTime(&ms, a, b);
        printf("N=%3d mode=%d (commit=%d wait=%d fence=%d): %.1f ns per k block (4 MMAs) = %.0f cycles  %s\n", n, mode, mode & 1, (mode >> 1) & 1, (mode >> 2) & 1,
               ms * 1e6 / groups, ms * 1e6 / groups * 1.965, cudaGetErrorString(cudaGetLastError()));
    }
    return 0;
}
