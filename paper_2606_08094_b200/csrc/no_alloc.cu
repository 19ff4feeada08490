// no_alloc.cu -- vla_ternary_linear_static: Eq. 4 end to end for callers that cannot allocate device
// memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The scratch that
// vla_ternary_linear needs -- the quantised activations a [M,K] int8 and their scales alpha [M] fp32, written by the
// activation quantiser and read by the GEMM kernel -- lives in ONE file-scope device array of fixed size instead of a
// caller-provided workspace.  Every GPU that loads the library holds the array (8.06 MiB) until the process exits.
//
// The array's name is a device symbol: in HOST code it is only a stand-in, not a device address.  Its address is looked up
// with cudaGetSymbolAddress, in this file, once per device, with that device current, and that pointer is what the kernels
// get.  Nothing here calls cudaMalloc / cudaFree or an allocating library routine.
//
// All calls share the array, and it keeps the last call's contents.  Nothing in it has to start at zero: the quantiser
// overwrites a[0 .. M*K) and alpha[0 .. M) of THIS call before the GEMM reads them (same stream, in order), and nothing
// beyond them is read.  Two calls that overlap on the GPU (different streams, or graphs replayed concurrently) RACE on it.
#include "../../include/vla_ternary.h"
#include <cstdint>
#include <mutex>
#include <cuda_runtime.h>

namespace {

constexpr size_t kMaxMK = (size_t)VLA_STATIC_MAX_MK;                // int8 elements of a [M,K]
constexpr size_t kMaxM = (size_t)VLA_STATIC_MAX_M;                  // rows (alpha)
constexpr size_t kAlphaOff = kMaxMK;                                // alpha [kMaxM] fp32 behind the int8 region
constexpr size_t kScratchBytes = kMaxMK + kMaxM * sizeof(float);
static_assert(kMaxMK % 256 == 0, "alpha must stay 256-byte aligned");

static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char* g_scratch_addr[kMaxDevices] = {};                    // per device: device address of g_static_scratch

// device address of the scratch array on the CURRENT device (looked up once per device)
cudaError_t scratch_of_current_device(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = reinterpret_cast<unsigned char*>(p);
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" vla_status vla_ternary_linear_static(const void* packed, const float* w_scale, const void* x_bf16,
                                                int M, int N, int K, void* out, vla_dtype out_dtype, vla_path path,
                                                void* stream) {
    if (!packed || !x_bf16 || !out) return VLA_ERR_NULL;
    if (M < 1 || N < 128 || K < 128) return VLA_ERR_SHAPE;
    // the fixed scratch bounds the problem: a [M,K] int8 and alpha [M] must fit
    if ((size_t)M > kMaxM || (size_t)M * (size_t)K > kMaxMK) return VLA_ERR_WORKSPACE;
    unsigned char* scratch = nullptr;
    if (scratch_of_current_device(&scratch) != cudaSuccess) {
        cudaGetLastError();
        return VLA_ERR_CUDA;
    }
    int8_t* xq = reinterpret_cast<int8_t*>(scratch);
    float* xs = reinterpret_cast<float*>(scratch + kAlphaOff);
    // the existing path, with its scratch pointed at the static array (no workspace, nothing allocated)
    return vla_ternary_linear(packed, w_scale, x_bf16, M, N, K, out, out_dtype, path, xq, xs, nullptr, 0, stream);
}
