// kernels.h -- host-side launchers of the CUDA kernels (internal to libvlaternary.so).
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

namespace vla {

// every launcher bumps this once per kernel it launches (vla_launch_count)
void count_launch(int n = 1);
unsigned long long launch_count();

cudaError_t launch_pack(const int8_t* w, int N, int K, void* packed, int* bad_flag, cudaStream_t s);
cudaError_t launch_unpack(const void* packed, int N, int K, int8_t* w, cudaStream_t s);
cudaError_t launch_act_quant(const void* x_bf16, int M, int K, int8_t* xq, float* x_scale, cudaStream_t s);

// out_dtype: 0 fp32, 1 bf16, 2 raw int32 (vla_dtype)
cudaError_t launch_gemm_small(bool use_mma, const void* packed, const float* w_scale, const int8_t* xq,
                              const float* x_scale, int M, int N, int K, void* out, int out_dtype, cudaStream_t s);
// up to 8 ternary linears that share one activation matrix, run as ONE tcgen05 launch (per-output-group scales)
struct LgGroup {
    const uint8_t* packed[8];
    const float* beta[8];
    void* out[8];
    int N[8];
    int dtype[8];
    int ct_begin[9];           // prefix sum of N / 128 (channel tiles)
    int n;
};
cudaError_t launch_gemm_large_grouped(const LgGroup& g, const int8_t* xq, const float* x_scale, int M, int K, cudaStream_t s);
cudaError_t launch_gemm_large(const void* packed, const float* w_scale, const int8_t* xq, const float* x_scale,
                              int M, int N, int K, void* out, int out_dtype, cudaStream_t s);
// persistent program kernel (gemm_program.cu); the program header travels as a kernel parameter
struct DevProg;
cudaError_t launch_program(const DevProg& prog, int grid, int max_m, cudaStream_t s);
cudaError_t program_max_ctas_per_sm(int max_m, int smem_bytes, int* out);      // co-residency of the persistent grid
cudaError_t run_i8_mma_probe(int ctas, int mmas_per_cta, float* ms_out);
// cached-conditioning cross-attention (attention.cu): d_k = 128, out_dtype 0 fp32 / 1 bf16
size_t attention_workspace_bytes(int Mq, int Mc, int Hq, int Hkv, int sms);
cudaError_t launch_attention(const void* q, const void* kc, const void* vc, const uint8_t* visible, int Mq, int Mc, int Hq,
                             int Hkv, void* out, int out_dtype, float* workspace, int sms, cudaStream_t s);

}  // namespace vla
