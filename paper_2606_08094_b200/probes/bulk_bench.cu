#include <cstdio>
#include "../csrc/common.cuh"
using namespace vla;
// each CTA streams `total` bytes from its own region through a ring of NS slots of SLOT bytes, `piece` bytes per bulk copy
__global__ void __launch_bounds__(64, 1) k(const uint8_t* src, size_t per_cta, int piece, int lanes_issue, long long* cyc) {
    extern __shared__ uint8_t smem_raw[];
    constexpr int NS = 10, SLOT = 16384;
    const uint32_t base = (smem_u32(smem_raw) + 127u) & ~127u;
    const uint32_t bar_full = base + NS * SLOT, bar_empty = bar_full + 8 * NS;
    if (threadIdx.x == 0) { for (int s = 0; s < NS; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, 1); } fence_barrier_init(); }
    __syncthreads();
    const uint8_t* my = src + (size_t)blockIdx.x * per_cta;
    const int nchunk = (int)(per_cta / SLOT), np = SLOT / piece;
    long long t0 = clock64();
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        for (int c = 0; c < nchunk; ++c) {
            const uint32_t s = c % NS;
            if (c >= NS) mbar_wait(bar_empty + 8 * s, ((c / NS) & 1) ^ 1);
            if (lane == 0) mbar_arrive_expect_tx(bar_full + 8 * s, SLOT);
            __syncwarp();
            if (lanes_issue) { for (int p = lane; p < np; p += 32) tma_bulk_g2s(base + s * SLOT + p * piece, my + (size_t)c * SLOT + (size_t)p * piece, piece, bar_full + 8 * s); }
            else if (lane == 0) { for (int p = 0; p < np; ++p) tma_bulk_g2s(base + s * SLOT + p * piece, my + (size_t)c * SLOT + (size_t)p * piece, piece, bar_full + 8 * s); }
        }
    } else if (threadIdx.x == 32) {
        for (int c = 0; c < nchunk; ++c) { const uint32_t s = c % NS; mbar_wait(bar_full + 8 * s, (c / NS) & 1); mbar_arrive(bar_empty + 8 * s); }
        if (blockIdx.x == 0) *cyc = clock64() - t0;
    }
}
int main() {
    const size_t per_cta = 4 << 20; const int ctas = 148;
    uint8_t* src; cudaMalloc(&src, per_cta * ctas); cudaMemset(src, 1, per_cta * ctas);
    long long* cyc; cudaMalloc(&cyc, 8);
    const int smem = 10 * 16384 + 512;
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    for (int li = 0; li < 2; ++li)
    for (int piece : {512, 1024, 2048, 4096, 16384}) {
        k<<<ctas, 64, smem>>>(src, per_cta, piece, li, cyc);
        cudaEventRecord(a); k<<<ctas, 64, smem>>>(src, per_cta, piece, li, cyc); cudaEventRecord(b); cudaDeviceSynchronize();
        float ms; cudaEventElapsedTime(&ms, a, b); long long h; cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
        printf("issue=%s piece=%5d: %.3f ms  %.0f GB/s total  (cta0: %.1f B/clk, %.0f cyc per 16KB chunk) %s\n", li ? "lanes" : "lane0", piece, ms, per_cta * ctas / ms / 1e6,
               (double)per_cta / h, (double)h / (per_cta / 16384), cudaGetErrorString(cudaGetLastError()));
    }
    return 0;
}
