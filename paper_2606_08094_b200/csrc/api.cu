// api.cu -- the C ABI of include/vla_ternary.h: host-side validation, path dispatch, status strings.
// Nothing here computes: every step of the path runs in the kernels of pack.cu, act_quant.cu,
// gemm_small.cu and gemm_large.cu.
#include "../../include/vla_ternary.h"
#include <atomic>
#include "kernels.h"

namespace vla {
static std::atomic<unsigned long long> g_launches{0};
void count_launch(int n) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }
unsigned long long launch_count() { return g_launches.load(std::memory_order_relaxed); }
}  // namespace vla

namespace {

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

inline bool shape_ok(int N, int K) { return N >= 128 && K >= 128 && N % 128 == 0 && K % 128 == 0 && K <= 65536; }

inline size_t round256(size_t b) { return (b + 255) / 256 * 256; }

vla_status check_arch() {                                  // per call: two cheap attribute queries, no cache to race on
    int dev = -1, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        cudaGetLastError();
        return VLA_ERR_ARCH;
    }
    return (major == 10) ? VLA_OK : VLA_ERR_ARCH;
}

inline vla_status from_cuda(cudaError_t e) {
    if (e == cudaSuccess) return VLA_OK;
    cudaGetLastError();
    return VLA_ERR_CUDA;
}

// The dispatch table: which kernel family runs a given M.
// Row a6.  M <= 16 and M > 32 are decided by M alone.  For 16 < M <= 32 both kernels run one token tile and
// neither is faster everywhere; measured on cold weights (profiles/r01d_path_probe.md): the IMMA kernel costs
// 7.5 us + 0.208 us per million weights, the tcgen05 kernel 4.1 us + 0.224 us per 128-wide k block per wave of
// 148 channel tiles.  The faster model wins.
vla_path auto_path(int M, int N, int K) {
    if (M <= 16) return VLA_PATH_SMALL_TC;
    if (M > 32) return VLA_PATH_LARGE;
    const double small_us = 7.5 + 0.208e-6 * (double)N * (double)K;
    const int waves = (N / 128 + 147) / 148;
    const double large_us = 4.1 + 0.224 * (double)(K / 128) * (double)waves;
    return large_us < small_us ? VLA_PATH_LARGE : VLA_PATH_SMALL_TC;
}

bool path_supports(vla_path p, int M) {
    switch (p) {
        case VLA_PATH_SMALL_ALU: return M <= 16;
        case VLA_PATH_SMALL_TC: return M <= 32;
        case VLA_PATH_LARGE: return true;
        default: return false;
    }
}

}  // namespace

extern "C" {

const char* vla_status_string(vla_status s) {
    switch (s) {
        case VLA_OK: return "VLA_OK";
        case VLA_ERR_NULL: return "VLA_ERR_NULL: a required pointer is NULL";
        case VLA_ERR_SHAPE: return "VLA_ERR_SHAPE: need M>=1, N%128==0, K%128==0, K<=65536; a forced path takes M<=16 (SMALL_ALU), M<=32 (SMALL_TC), any M (LARGE)";
        case VLA_ERR_ALIGN: return "VLA_ERR_ALIGN: pointers must be 16-byte aligned";
        case VLA_ERR_VALUE: return "VLA_ERR_VALUE: weight element outside {-1,0,+1}, or not a compiled program";
        case VLA_ERR_DTYPE: return "VLA_ERR_DTYPE: unknown vla_dtype or vla_path";
        case VLA_ERR_WORKSPACE: return "VLA_ERR_WORKSPACE: workspace missing or too small";
        case VLA_ERR_ARCH: return "VLA_ERR_ARCH: current device is not sm_100 (no fallback path exists)";
        case VLA_ERR_CUDA: return "VLA_ERR_CUDA: CUDA runtime/driver error";
    }
    return "unknown vla_status";
}

size_t vla_ternary_packed_bytes(int N, int K) {
    if (!shape_ok(N, K)) return 0;
    return (size_t)N * (size_t)K / 4;
}

size_t vla_ternary_workspace_bytes(int M, int N, int K, vla_path path) {
    (void)path;
    if (M < 1 || !shape_ok(N, K)) return 0;
    // room for the quantised activations of vla_ternary_linear: int8 [M,K] + fp32 [M]
    return round256((size_t)M * K) + round256((size_t)M * 4);
}

vla_path vla_ternary_auto_path(int M, int N, int K) {
    return auto_path(M, N, K);
}

vla_status vla_ternary_pack(const int8_t* w, int N, int K, void* packed, size_t packed_bytes, void* stream) {
    if (!w || !packed) return VLA_ERR_NULL;
    if (!shape_ok(N, K)) return VLA_ERR_SHAPE;
    if (packed_bytes < vla_ternary_packed_bytes(N, K)) return VLA_ERR_WORKSPACE;       // the documented code for a short buffer
    if (!aligned16(w) || !aligned16(packed)) return VLA_ERR_ALIGN;
    vla_status st = check_arch();
    if (st != VLA_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    int* flag = nullptr;
    if (cudaMallocAsync(&flag, sizeof(int), s) != cudaSuccess) return from_cuda(cudaErrorMemoryAllocation);
    int host_flag = 0;
    cudaError_t e = cudaMemsetAsync(flag, 0, sizeof(int), s);
    if (e == cudaSuccess) e = vla::launch_pack(w, N, K, packed, flag, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&host_flag, flag, sizeof(int), cudaMemcpyDeviceToHost, s);
    cudaFreeAsync(flag, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return from_cuda(e);
    return host_flag ? VLA_ERR_VALUE : VLA_OK;
}

vla_status vla_ternary_unpack(const void* packed, int N, int K, int8_t* w, void* stream) {
    if (!w || !packed) return VLA_ERR_NULL;
    if (!shape_ok(N, K)) return VLA_ERR_SHAPE;
    if (!aligned16(w) || !aligned16(packed)) return VLA_ERR_ALIGN;
    vla_status st = check_arch();
    if (st != VLA_OK) return st;
    return from_cuda(vla::launch_unpack(packed, N, K, w, (cudaStream_t)stream));
}

vla_status vla_act_quant(const void* x_bf16, int M, int K, int8_t* xq, float* x_scale, void* stream) {
    if (!x_bf16 || !xq || !x_scale) return VLA_ERR_NULL;
    if (M < 1 || K < 128 || K % 128 != 0 || K > 65536) return VLA_ERR_SHAPE;
    if (!aligned16(x_bf16) || !aligned16(xq) || !aligned16(x_scale)) return VLA_ERR_ALIGN;
    vla_status st = check_arch();
    if (st != VLA_OK) return st;
    return from_cuda(vla::launch_act_quant(x_bf16, M, K, xq, x_scale, (cudaStream_t)stream));
}

vla_status vla_ternary_gemm(const void* packed, const float* w_scale, const int8_t* xq, const float* x_scale,
                            int M, int N, int K, void* out, vla_dtype out_dtype, vla_path path,
                            void* workspace, size_t workspace_bytes, void* stream) {
    (void)workspace; (void)workspace_bytes;           // no GEMM path needs scratch at present
    if ((int)out_dtype < 0 || (int)out_dtype > 2 || (int)path < 0 || (int)path > 3) return VLA_ERR_DTYPE;
    if (!packed || !xq || !out) return VLA_ERR_NULL;
    if (out_dtype != VLA_I32 && (!w_scale || !x_scale)) return VLA_ERR_NULL;
    if (M < 1 || !shape_ok(N, K)) return VLA_ERR_SHAPE;
    if (path == VLA_PATH_AUTO) path = auto_path(M, N, K);
    if (!path_supports(path, M)) return VLA_ERR_SHAPE;
    if (!aligned16(packed) || !aligned16(xq) || !aligned16(out) || (x_scale && !aligned16(x_scale)) ||
        (w_scale && (reinterpret_cast<uintptr_t>(w_scale) & 3u)))
        return VLA_ERR_ALIGN;
    vla_status st = check_arch();
    if (st != VLA_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e;
    if (path == VLA_PATH_LARGE)
        e = vla::launch_gemm_large(packed, w_scale, xq, x_scale, M, N, K, out, (int)out_dtype, s);
    else
        e = vla::launch_gemm_small(path == VLA_PATH_SMALL_TC, packed, w_scale, xq, x_scale, M, N, K, out, (int)out_dtype, s);
    return from_cuda(e);
}

vla_status vla_ternary_linear(const void* packed, const float* w_scale, const void* x_bf16,
                              int M, int N, int K, void* out, vla_dtype out_dtype, vla_path path,
                              int8_t* xq_opt, float* x_scale_opt,
                              void* workspace, size_t workspace_bytes, void* stream) {
    if (!x_bf16) return VLA_ERR_NULL;
    if (M < 1 || !shape_ok(N, K)) return VLA_ERR_SHAPE;
    int8_t* xq = xq_opt;
    float* xs = x_scale_opt;
    if (!xq || !xs) {
        if (!workspace || workspace_bytes < vla_ternary_workspace_bytes(M, N, K, path)) return VLA_ERR_WORKSPACE;
        if (!aligned16(workspace)) return VLA_ERR_ALIGN;
        if (!xq) xq = reinterpret_cast<int8_t*>(workspace);
        if (!xs) xs = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(workspace) + round256((size_t)M * K));
    }
    // validate the GEMM's arguments before launching anything
    if ((int)out_dtype < 0 || (int)out_dtype > 2 || (int)path < 0 || (int)path > 3) return VLA_ERR_DTYPE;
    if (!packed || !out || (out_dtype != VLA_I32 && !w_scale)) return VLA_ERR_NULL;
    if (path != VLA_PATH_AUTO && !path_supports(path, M)) return VLA_ERR_SHAPE;
    if (!aligned16(packed) || !aligned16(out) || !aligned16(x_bf16) || !aligned16(xq) || !aligned16(xs)) return VLA_ERR_ALIGN;
    vla_status st = vla_act_quant(x_bf16, M, K, xq, xs, stream);
    if (st != VLA_OK) return st;
    return vla_ternary_gemm(packed, w_scale, xq, xs, M, N, K, out, out_dtype, path, nullptr, 0, stream);
}

size_t vla_ternary_host_workspace_bytes(int M, int N, int K, vla_dtype out_dtype, vla_path path) {
    size_t inner = vla_ternary_workspace_bytes(M, N, K, path);
    if (inner == 0 || (int)out_dtype < 0 || (int)out_dtype > 2) return 0;
    size_t esz = (out_dtype == VLA_BF16) ? 2 : 4;
    return inner + round256((size_t)M * K * 2) + round256((size_t)M * N * esz);
}

vla_status vla_ternary_linear_host(const void* packed, const float* w_scale, const void* x_bf16_host,
                                   int M, int N, int K, void* out_host, vla_dtype out_dtype, vla_path path,
                                   void* workspace, size_t workspace_bytes, void* stream) {
    if (!x_bf16_host || !out_host) return VLA_ERR_NULL;
    if ((int)out_dtype < 0 || (int)out_dtype > 2 || (int)path < 0 || (int)path > 3) return VLA_ERR_DTYPE;
    if (M < 1 || !shape_ok(N, K)) return VLA_ERR_SHAPE;
    const size_t need = vla_ternary_host_workspace_bytes(M, N, K, out_dtype, path);
    if (!workspace || workspace_bytes < need) return VLA_ERR_WORKSPACE;
    if (!aligned16(workspace)) return VLA_ERR_ALIGN;
    const size_t inner = vla_ternary_workspace_bytes(M, N, K, path);
    const size_t xbytes = (size_t)M * K * 2, obytes = (size_t)M * N * ((out_dtype == VLA_BF16) ? 2 : 4);
    uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
    void* x_dev = ws + inner;
    void* out_dev = ws + inner + round256(xbytes);
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(x_dev, x_bf16_host, xbytes, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return from_cuda(e);
    vla_status st = vla_ternary_linear(packed, w_scale, x_dev, M, N, K, out_dev, out_dtype, path, nullptr, nullptr,
                                       workspace, inner, stream);
    if (st != VLA_OK) return st;
    e = cudaMemcpyAsync(out_host, out_dev, obytes, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    return from_cuda(e);
}

// ---------------------------------------------------------------- cached-conditioning attention (Eq. 2)
static bool attn_shape_ok(int Mq, int Mc, int Hq, int Hkv, int d_k) {
    return Mq >= 1 && Mq <= 4096 && Mc >= 1 && Mc <= 65536 && d_k == 128 && Hkv >= 1 && Hq >= Hkv && Hq % Hkv == 0 &&
           Hq / Hkv <= 8 && Hq <= 1024;
}
static int current_sms() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return 148;                                           // (sizes only; the launch itself reports the error)
    }
    return sms > 0 ? sms : 148;
}

size_t vla_cached_attention_workspace_bytes(int Mq, int Mc, int n_q_heads, int n_kv_heads, int d_k) {
    if (!attn_shape_ok(Mq, Mc, n_q_heads, n_kv_heads, d_k)) return 0;
    // sized for the most splits any device takes (one per 64-key tile), so the answer does not depend on the device
    return round256((size_t)((Mc + 63) / 64) * n_q_heads * Mq * (128 + 2) * sizeof(float));
}

vla_status vla_cached_attention(const void* q_bf16, const void* kc_bf16, const void* vc_bf16, const uint8_t* visible_opt,
                                int Mq, int Mc, int n_q_heads, int n_kv_heads, int d_k, void* out, vla_dtype out_dtype,
                                void* workspace, size_t workspace_bytes, void* stream) {
    if (!q_bf16 || !kc_bf16 || !vc_bf16 || !out) return VLA_ERR_NULL;
    if (out_dtype != VLA_F32 && out_dtype != VLA_BF16) return VLA_ERR_DTYPE;
    if (!attn_shape_ok(Mq, Mc, n_q_heads, n_kv_heads, d_k)) return VLA_ERR_SHAPE;
    if (!aligned16(q_bf16) || !aligned16(kc_bf16) || !aligned16(vc_bf16) || !aligned16(out)) return VLA_ERR_ALIGN;
    vla_status st = check_arch();
    if (st != VLA_OK) return st;
    const int sms = current_sms();
    const size_t need = vla::attention_workspace_bytes(Mq, Mc, n_q_heads, n_kv_heads, sms);
    if (need > 0) {
        if (!workspace || workspace_bytes < need) return VLA_ERR_WORKSPACE;
        if (!aligned16(workspace)) return VLA_ERR_ALIGN;
    }
    return from_cuda(vla::launch_attention(q_bf16, kc_bf16, vc_bf16, visible_opt, Mq, Mc, n_q_heads, n_kv_heads, out,
                                           (int)out_dtype, reinterpret_cast<float*>(workspace), sms, (cudaStream_t)stream));
}

unsigned long long vla_launch_count(void) { return vla::launch_count(); }

vla_status vla_i8_mma_issue_probe(int ctas, int mmas_per_cta, float* ms_out) {
    if (!ms_out) return VLA_ERR_NULL;
    if (ctas < 1 || mmas_per_cta < 1) return VLA_ERR_SHAPE;
    vla_status st = check_arch();
    if (st != VLA_OK) return st;
    return from_cuda(vla::run_i8_mma_probe(ctas, mmas_per_cta, ms_out));
}

}  // extern "C"
