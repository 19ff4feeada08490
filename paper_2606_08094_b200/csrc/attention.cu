// attention.cu -- cached-conditioning cross-attention, Eq. 2 of the paper (section III-B):
//     Attn(Q, K_C, V_C; M) = softmax(Q K_C^T / sqrt(d_k) + M) V_C        (one head; softmax over keys)
// K_C = Z W_K and V_C = Z W_V are the CACHED projections of the conditioning sequence: they are computed once per
// observation (here: by the k / v ternary linears of Eq. 4) and reused by every solver step, so a step reads them from L2.
//
// The action-query side is small (M_q = the action chunk, <= 16 rows per pass) and the conditioning side is a few hundred
// keys: the call is latency-bound, so the work is split flash-decoding style over as many CTAs as there are SMs:
//   grid = (key splits, KV heads, query tiles of 16 rows); one WARP per query head of the KV head's group (grouped-query
//   attention, R14: query head h reads KV head h / (Hq / Hkv)), so a K / V tile staged in shared memory is
//   shared by the whole group.
//   per 64-key tile:  S = Q K^T on the warp-level bf16 MMA (m16n8k16, fp32 accumulation: bf16 x bf16 products are exact in
//   fp32), mask, online softmax in fp32 (exp2 with log2(e)/sqrt(d_k) folded in), then  O += P V  again on the MMA with
//   P split into two bf16 terms (hi + lo, |P - hi - lo| <= 2^-17 P) so that the probabilities are NOT rounded to bf16.
//   Partial (O, row max, row sum) per split -> workspace; attn_combine_kernel merges the splits and normalises.
// Rows whose keys are all masked give 0 (R15).  tcgen05 is not used: its MMA needs 64 / 128 rows per instruction, a
// 16-row action chunk would waste 3/4 of it, and nothing here is tensor-bound.
#include <cuda_bf16.h>
#include <math_constants.h>
#include "common.cuh"
#include "kernels.h"

namespace vla {

constexpr int AT_D = 128;                        // head dimension (BASELINE.json configs[3])
constexpr int AT_KT = 64;                        // keys per tile
constexpr int AT_KROW = AT_D + 8;                // padded K row (bf16): 272 B, conflict-free fragment loads
constexpr int AT_VROW = AT_KT + 8;               // padded V^T row (bf16): 144 B
constexpr int AT_MAXG = 8;                       // query heads per KV head

__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    return (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(lo)) | ((uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(hi)) << 16);
}
__device__ __forceinline__ float bf16_round(float x) { return __bfloat162float(__float2bfloat16_rn(x)); }

// One CTA: KV head blockIdx.y, query rows [16 * blockIdx.z, +16), keys [k_begin, k_end) of split blockIdx.x.
// part: [split][q head][Mq rows][AT_D + 2] fp32 = unnormalised O, running max (in units of the raw score), running sum.
__global__ void __launch_bounds__(AT_MAXG * 32, 1) attn_partial_kernel(
    const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ kc, const __nv_bfloat16* __restrict__ vc,
    const uint8_t* __restrict__ visible, int Mq, int Mc, int Hq, int Hkv, int keys_per_split, float* __restrict__ part,
    void* __restrict__ out, int out_dtype, int n_splits) {
    __shared__ __align__(16) __nv_bfloat16 sK[AT_KT * AT_KROW];
    __shared__ __align__(16) __nv_bfloat16 sVt[AT_D * AT_VROW];
    const int group = Hq / Hkv, warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int kvh = blockIdx.y, h = kvh * group + warp, m0 = blockIdx.z * 16;
    const int k_begin = blockIdx.x * keys_per_split, k_end = min(Mc, k_begin + keys_per_split);
    const float c = 1.4426950408889634f * rsqrtf((float)AT_D);      // log2(e) / sqrt(d_k): p = exp2((s - max) * c)
    pdl_wait();                                               // q (and, on the first step, K_C / V_C) come from earlier kernels

    // Q fragments of this warp's head: rows m0+g and m0+g+8, all 128 d (zero rows beyond Mq)
    uint32_t qa[AT_D / 16][4];
    {
        const int r0 = m0 + g, r1 = m0 + g + 8;
        const uint32_t* q0 = reinterpret_cast<const uint32_t*>(q + (size_t)r0 * Hq * AT_D + h * AT_D);
        const uint32_t* q1 = reinterpret_cast<const uint32_t*>(q + (size_t)r1 * Hq * AT_D + h * AT_D);
#pragma unroll
        for (int ks = 0; ks < AT_D / 16; ++ks) {
            qa[ks][0] = r0 < Mq ? q0[ks * 8 + t] : 0u;
            qa[ks][1] = r1 < Mq ? q1[ks * 8 + t] : 0u;
            qa[ks][2] = r0 < Mq ? q0[ks * 8 + 4 + t] : 0u;
            qa[ks][3] = r1 < Mq ? q1[ks * 8 + 4 + t] : 0u;
        }
    }
    float o[AT_D / 8][4];
#pragma unroll
    for (int nd = 0; nd < AT_D / 8; ++nd) o[nd][0] = o[nd][1] = o[nd][2] = o[nd][3] = 0.0f;
    float m_run[2] = {-CUDART_INF_F, -CUDART_INF_F}, l_run[2] = {0.0f, 0.0f};

    for (int k0 = k_begin; k0 < k_end; k0 += AT_KT) {
        __syncthreads();                                      // the previous tile has been consumed
        // K tile: 16-byte chunks, row-major, padded rows; keys beyond Mc are zero
        for (int idx = threadIdx.x; idx < AT_KT * (AT_D / 8); idx += blockDim.x) {
            const int key = idx / (AT_D / 8), ch = idx % (AT_D / 8);
            uint4 v = make_uint4(0, 0, 0, 0);
            if (k0 + key < k_end) v = *reinterpret_cast<const uint4*>(kc + (size_t)(k0 + key) * Hkv * AT_D + kvh * AT_D + ch * 8);
            *reinterpret_cast<uint4*>(sK + key * AT_KROW + ch * 8) = v;
        }
        // V tile, transposed to [d][key]: a lane owns a key, so the 32 two-byte stores of a warp are contiguous
        for (int idx = threadIdx.x; idx < AT_KT * (AT_D / 8); idx += blockDim.x) {
            const int key = (idx & 31) + 32 * ((idx >> 5) % (AT_KT / 32)), ch = (idx >> 5) / (AT_KT / 32);
            uint4 v = make_uint4(0, 0, 0, 0);
            if (k0 + key < k_end) v = *reinterpret_cast<const uint4*>(vc + (size_t)(k0 + key) * Hkv * AT_D + kvh * AT_D + ch * 8);
            const uint32_t w4[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int i = 0; i < 8; ++i)
                reinterpret_cast<unsigned short*>(sVt)[(ch * 8 + i) * AT_VROW + key] = (unsigned short)(w4[i >> 1] >> (16 * (i & 1)));
        }
        __syncthreads();
        if (warp < group) {
            // S = Q K^T for the 64 keys of the tile: 8 n-tiles of 8 keys
            float s[AT_KT / 8][4];
#pragma unroll
            for (int nt = 0; nt < AT_KT / 8; ++nt) {
                s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.0f;
                const uint32_t* kr = reinterpret_cast<const uint32_t*>(sK + (nt * 8 + g) * AT_KROW);
#pragma unroll
                for (int ks = 0; ks < AT_D / 16; ++ks)
                    mma_bf16_16816(s[nt], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], kr[ks * 8 + t], kr[ks * 8 + 4 + t]);
            }
            // + M: keys beyond the range and masked keys are -inf
            float tmax[2] = {-CUDART_INF_F, -CUDART_INF_F};
#pragma unroll
            for (int nt = 0; nt < AT_KT / 8; ++nt)
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int key = k0 + nt * 8 + 2 * t + (i & 1), row = m0 + g + 8 * (i >> 1);
                    bool vis = key < k_end && row < Mq;
                    if (vis && visible != nullptr) vis = visible[(size_t)row * Mc + key] != 0;
                    if (!vis) s[nt][i] = -CUDART_INF_F;
                    tmax[i >> 1] = fmaxf(tmax[i >> 1], s[nt][i]);
                }
            float scale[2], m_use[2];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                tmax[r] = fmaxf(tmax[r], __shfl_xor_sync(0xFFFFFFFFu, tmax[r], 1));
                tmax[r] = fmaxf(tmax[r], __shfl_xor_sync(0xFFFFFFFFu, tmax[r], 2));
                const float m_new = fmaxf(m_run[r], tmax[r]);
                m_use[r] = (m_new == -CUDART_INF_F) ? 0.0f : m_new;            // nothing visible yet: exponents of -inf
                scale[r] = exp2f((m_run[r] - m_use[r]) * c);                    // (m_run = -inf -> 0)
                m_run[r] = m_new;
                l_run[r] *= scale[r];
            }
#pragma unroll
            for (int nd = 0; nd < AT_D / 8; ++nd) {
                o[nd][0] *= scale[0]; o[nd][1] *= scale[0];
                o[nd][2] *= scale[1]; o[nd][3] *= scale[1];
            }
            // P = exp2((S - max) c), its row sums, and O += P V with P = hi + lo in bf16
#pragma unroll
            for (int kk = 0; kk < AT_KT / 16; ++kk) {
                float p[2][4];
#pragma unroll
                for (int j = 0; j < 2; ++j)
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        p[j][i] = exp2f((s[2 * kk + j][i] - m_use[i >> 1]) * c);
                        l_run[i >> 1] += p[j][i];
                    }
                uint32_t ah[4], al[4];
#pragma unroll
                for (int j = 0; j < 2; ++j)
#pragma unroll
                    for (int r = 0; r < 2; ++r) {
                        const float x0 = p[j][2 * r], x1 = p[j][2 * r + 1];
                        const float h0 = bf16_round(x0), h1 = bf16_round(x1);
                        ah[2 * j + r] = pack_bf16(h0, h1);
                        al[2 * j + r] = pack_bf16(x0 - h0, x1 - h1);
                    }
#pragma unroll
                for (int nd = 0; nd < AT_D / 8; ++nd) {
                    const uint32_t* vr = reinterpret_cast<const uint32_t*>(sVt + (nd * 8 + g) * AT_VROW + kk * 16);
                    const uint32_t b0 = vr[t], b1 = vr[4 + t];
                    mma_bf16_16816(o[nd], ah[0], ah[1], ah[2], ah[3], b0, b1);
                    mma_bf16_16816(o[nd], al[0], al[1], al[2], al[3], b0, b1);
                }
            }
        }
    }
    pdl_launch_dependents();
    if (warp >= group) return;
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        l_run[r] += __shfl_xor_sync(0xFFFFFFFFu, l_run[r], 1);
        l_run[r] += __shfl_xor_sync(0xFFFFFFFFu, l_run[r], 2);
    }
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int row = m0 + g + 8 * r;
        if (row >= Mq) continue;
        if (n_splits == 1) {                                  // no merge needed: normalise and store
            const float inv = l_run[r] > 0.0f ? __fdiv_rn(1.0f, l_run[r]) : 0.0f;      // R15: all keys masked -> 0
            const size_t ob = (size_t)row * Hq * AT_D + h * AT_D + 2 * t;
#pragma unroll
            for (int nd = 0; nd < AT_D / 8; ++nd) {
                const float y0 = o[nd][2 * r] * inv, y1 = o[nd][2 * r + 1] * inv;
                if (out_dtype == 0) *reinterpret_cast<float2*>(reinterpret_cast<float*>(out) + ob + nd * 8) = make_float2(y0, y1);
                else *reinterpret_cast<uint32_t*>(reinterpret_cast<__nv_bfloat16*>(out) + ob + nd * 8) = pack_bf16(y0, y1);
            }
        } else {
            float* pr = part + (((size_t)blockIdx.x * Hq + h) * Mq + row) * (AT_D + 2);
#pragma unroll
            for (int nd = 0; nd < AT_D / 8; ++nd)
                *reinterpret_cast<float2*>(pr + nd * 8 + 2 * t) = make_float2(o[nd][2 * r], o[nd][2 * r + 1]);
            if (t == 0) { pr[AT_D] = m_run[r]; pr[AT_D + 1] = l_run[r]; }
        }
    }
}

// merge the key splits of one (row, head): out = sum_s O_s 2^((m_s - m) c) / sum_s l_s 2^((m_s - m) c)
__global__ void __launch_bounds__(AT_D) attn_combine_kernel(const float* __restrict__ part, int Mq, int Hq, int n_splits,
                                                            void* __restrict__ out, int out_dtype) {
    const int row = blockIdx.x, h = blockIdx.y, d = threadIdx.x;
    const float c = 1.4426950408889634f * rsqrtf((float)AT_D);
    pdl_wait();
    float m = -CUDART_INF_F;
    for (int s = 0; s < n_splits; ++s) m = fmaxf(m, part[(((size_t)s * Hq + h) * Mq + row) * (AT_D + 2) + AT_D]);
    float acc = 0.0f, l = 0.0f;
    if (m != -CUDART_INF_F)
        for (int s = 0; s < n_splits; ++s) {
            const float* pr = part + (((size_t)s * Hq + h) * Mq + row) * (AT_D + 2);
            const float w = exp2f((pr[AT_D] - m) * c);         // (a split with nothing visible: m_s = -inf -> 0)
            acc += pr[d] * w;
            l += pr[AT_D + 1] * w;
        }
    pdl_launch_dependents();
    const float y = l > 0.0f ? __fdiv_rn(acc, l) : 0.0f;       // R15
    const size_t o = (size_t)row * Hq * AT_D + h * AT_D + d;
    if (out_dtype == 0) reinterpret_cast<float*>(out)[o] = y;
    else reinterpret_cast<__nv_bfloat16*>(out)[o] = __float2bfloat16_rn(y);
}

int attention_splits(int Mq, int Mc, int Hkv, int sms) {
    const int q_tiles = (Mq + 15) / 16, tiles = (Mc + AT_KT - 1) / AT_KT;
    int s = sms / (Hkv * q_tiles);
    if (s < 1) s = 1;
    return s < tiles ? s : tiles;
}

size_t attention_workspace_bytes(int Mq, int Mc, int Hq, int Hkv, int sms) {
    const int s = attention_splits(Mq, Mc, Hkv, sms);
    return s == 1 ? 0 : (size_t)s * Hq * Mq * (AT_D + 2) * sizeof(float);
}

cudaError_t launch_attention(const void* q, const void* kc, const void* vc, const uint8_t* visible, int Mq, int Mc, int Hq,
                             int Hkv, void* out, int out_dtype, float* workspace, int sms, cudaStream_t s) {
    const int n_splits = attention_splits(Mq, Mc, Hkv, sms);
    const int tiles = (Mc + AT_KT - 1) / AT_KT;
    const int keys_per_split = ((tiles + n_splits - 1) / n_splits) * AT_KT;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_splits, (unsigned)Hkv, (unsigned)((Mq + 15) / 16));
    cfg.blockDim = dim3((unsigned)(max(4, Hq / Hkv) * 32));
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    count_launch();
    cudaError_t e = cudaLaunchKernelEx(&cfg, attn_partial_kernel, (const __nv_bfloat16*)q, (const __nv_bfloat16*)kc,
                                       (const __nv_bfloat16*)vc, visible, Mq, Mc, Hq, Hkv, keys_per_split, workspace, out,
                                       out_dtype, n_splits);
    if (e != cudaSuccess || n_splits == 1) return e;
    cfg.gridDim = dim3((unsigned)Mq, (unsigned)Hq);
    cfg.blockDim = dim3(AT_D);
    count_launch();
    return cudaLaunchKernelEx(&cfg, attn_combine_kernel, (const float*)workspace, Mq, Hq, n_splits, out, out_dtype);
}

}  // namespace vla
