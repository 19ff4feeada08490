#include <cstdio>
#include "../csrc/common.cuh"
using namespace vla;
__global__ void __launch_bounds__(64, 1) probe(int iters, int n, int distinct) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* base_ptr = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t sA = base, sB = base + 4 * 16384, sBar = sB + 4 * 32768;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < (4 * 16384 + 4 * 32768) / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(base_ptr)[i] = 0x01010101u;
    fence_proxy_async_smem();
    if (threadIdx.x == 0) { mbar_init(sBar, 1); fence_barrier_init(); }
    if (warp == 1) tmem_alloc(sBar + 8, 256);
    tc_fence_before(); __syncthreads(); tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(base_ptr + 4 * 16384 + 4 * 32768 + 8);
    if (warp == 0 && lane == 0) {
        const uint32_t idesc = umma_idesc_i8(128, n);
        for (int i = 0; i < iters; ++i) {
            int st = distinct ? ((i >> 2) & 3) : 0;
            const uint64_t a = umma_desc_k_sw128(sA + st * 16384), b = umma_desc_k_sw128(sB + st * 32768);
            mma_i8_ss(tmem_base, a + 2 * (i & 3), b + 2 * (i & 3), idesc, i != 0);
        }
        mma_commit(sBar); mbar_wait(sBar, 0);
    }
    tc_fence_before(); __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, 256);
}
int main() {
    const int smem = 4 * 16384 + 4 * 32768 + 1024 + 64;
    cudaFuncSetAttribute(probe, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    const int iters = 20000;
    for (int distinct = 0; distinct < 2; ++distinct)
    for (int n : {16, 48, 96, 128, 192, 256}) {
        probe<<<148, 64, smem>>>(iters, n, distinct);
        cudaEventRecord(a); probe<<<148, 64, smem>>>(iters, n, distinct); cudaEventRecord(b); cudaDeviceSynchronize();
        float ms; cudaEventElapsedTime(&ms, a, b);
        printf("distinct=%d N=%3d: %.1f ns per MMA  (%.0f TOPS)  %s\n", distinct, n, ms * 1e6 / iters, 2.0 * 128 * n * 32 * iters * 148 / ms / 1e9, cudaGetErrorString(cudaGetLastError()));
    }
    return 0;
}
