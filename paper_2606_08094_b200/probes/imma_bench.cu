#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
__device__ __forceinline__ void mma_s8(int (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
template <int CHAINS>
__global__ void k_imma(int iters, int* out, long long* cyc) {
    int c[CHAINS][4] = {};
    uint32_t a = threadIdx.x * 0x01010101u, b = 0x01020304u;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < CHAINS; ++j) mma_s8(c[j], a, a + j, a ^ 5, a + 7, b, b + j);
    }
    long long t1 = clock64();
    int s = 0;
    for (int j = 0; j < CHAINS; ++j) s += c[j][0] + c[j][1] + c[j][2] + c[j][3];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}
template <int CHAINS>
__global__ void k_dp4a(int iters, int* out, long long* cyc) {
    int c[CHAINS] = {};
    int a = threadIdx.x * 0x01010101, b = 0x01020304;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < CHAINS; ++j) c[j] = __dp4a(a + j, b, c[j]);
    }
    long long t1 = clock64();
    int s = 0;
    for (int j = 0; j < CHAINS; ++j) s += c[j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}
int main() {
    int* out; long long* cyc; cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&cyc, 8);
    long long h;
    const int iters = 4096;
    for (int warps : {1, 4, 8, 16}) {
        k_imma<1><<<148, warps * 32>>>(iters, out, cyc); cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
        printf("IMMA warps/SM=%2d chains=1: %.2f cyc per IMMA per warp (latency-bound if 1 warp/SP)\n", warps, (double)h / iters);
        k_imma<8><<<148, warps * 32>>>(iters, out, cyc); cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
        printf("IMMA warps/SM=%2d chains=8: %.2f cyc per IMMA per warp -> %.2f cyc per IMMA per SP\n", warps, (double)h / iters / 8,
               (double)h / iters / 8 / ((warps + 3) / 4));
    }
    for (int warps : {4, 16}) {
        k_dp4a<8><<<148, warps * 32>>>(iters, out, cyc); cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
        printf("DP4A warps/SM=%2d chains=8: %.2f cyc per warp-instr per warp -> %.2f per SP\n", warps, (double)h / iters / 8, (double)h / iters / 8 / ((warps + 3) / 4));
    }
    printf("err %s\n", cudaGetErrorString(cudaDeviceSynchronize()));
    return 0;
}
