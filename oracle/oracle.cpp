// oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU restatement of the ternary linear layer of
// arxiv/paper_2606_08094 ("vla.cpp"), Section III-D, Eq. 4:
//
//     alpha_m = max(||x_m||_inf, 1e-5) / 127                      (Eq. 4, line 1)
//     a_mj    = clip_[-128,127]( round( x_mj / alpha_m ) )        (Eq. 4, line 2)
//     y_mn    = alpha_m * beta_g(n) * sum_j a_mj q_nj             (Eq. 4, line 3)
//
// "Products accumulate in 32-bit integers and are scaled to bfloat16 ... Rounding uses
// nearest-even ties; the output equation describes the scaled product before BF16
// conversion."
//
// Every function below executes that definition one scalar operation at a time, in IEEE-754
// binary32 where the paper's arithmetic is floating point, over UNPACKED int8 weights.
// It shares no code, header, table or helper with the CUDA library under
// paper_2606_08094_b200/ and neither imports the other.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may load it.
//
// Readings of the paper where it is silent or ambiguous are listed in DESIGN.md ("Readings");
// the ones that touch this file:
//   R1  x/alpha and max(.)/127 are true fp32 divisions (round-to-nearest), not reciprocal multiplies.
//   R2  clip range: the paper writes [-128,127]; with R1 the value -128 is unreachable for finite
//       input, so the clamp used is [-127,127] (BASELINE.json north_star: "clamp +-127").
//   R3  "round" = round-half-to-even (P:L82 applies to both the activation rounding and BF16).
//   R4  1e-5 is the fp32 constant 1e-5f.
//   R6  y = (float)acc * (alpha_m * beta): alpha*beta first (one fp32 multiply), then one multiply.
//   R7  beta_g(n): one output group (one scale per tensor); the grouped form takes a [G] vector.
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): exact-rational brute force on tiny shapes,
// exhaustive 3^(N*K) weight patterns, the worked vector in tests/golden/, unit-vector / all-ones /
// negation invariants, numpy/BLAS integer matmul at full size, quantiser invariants, torch bf16 cast.
// No function here is "parity unpinned".
//
// Build: g++ -O3 -march=native -fopenmp -fno-fast-math -ffp-contract=off -shared -fPIC

#include <cfenv>
#include <cmath>
#include <cstdint>
#include <cstring>

#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// O1: bf16 -> fp32 is exact: the 16 stored bits are the top half of the binary32 pattern.
static inline float bf16_bits_to_f32(uint16_t b) {
    uint32_t u = (uint32_t)b << 16;
    float f;
    std::memcpy(&f, &u, 4);
    return f;
}

void orc_bf16_to_f32(const uint16_t* x, long n, float* out) {
    for (long i = 0; i < n; ++i) out[i] = bf16_bits_to_f32(x[i]);
}

// O7: fp32 -> bf16 with round-to-nearest, ties to even.  Finite inputs only.
static inline uint16_t f32_to_bf16_rne(float f) {
    uint32_t u;
    std::memcpy(&u, &f, 4);
    uint32_t lsb = (u >> 16) & 1u;      // the bit that becomes the bf16 LSB
    u += 0x7FFFu + lsb;                  // half-ulp minus one, plus one when the LSB is odd
    return (uint16_t)(u >> 16);
}

void orc_f32_to_bf16(const float* x, long n, uint16_t* out) {
    for (long i = 0; i < n; ++i) out[i] = f32_to_bf16_rne(x[i]);
}

// O2-O4 (Eq. 4 lines 1-2): per-row absmax int8 quantisation of a bf16 activation matrix.
//   x      [M,K] bf16 bit patterns, row-major
//   a      [M,K] int8
//   alpha  [M]   fp32
void orc_act_quant(const uint16_t* x, int M, int K, int8_t* a, float* alpha) {
    std::fesetround(FE_TONEAREST);
    for (int m = 0; m < M; ++m) {
        const uint16_t* xr = x + (long)m * K;
        float amax = 0.0f;                                   // O2: ||x_m||_inf
        for (int j = 0; j < K; ++j) {
            float v = std::fabs(bf16_bits_to_f32(xr[j]));
            if (v > amax) amax = v;
        }
        float al = std::fmax(amax, 1e-5f) / 127.0f;          // O3: one fp32 division
        alpha[m] = al;
        for (int j = 0; j < K; ++j) {
            float t = bf16_bits_to_f32(xr[j]) / al;          // O4: one fp32 division
            float r = std::nearbyintf(t);                    //     ties to even
            if (r > 127.0f) r = 127.0f;                      //     clamp (R2)
            if (r < -127.0f) r = -127.0f;
            a[(long)m * K + j] = (int8_t)r;
        }
    }
}

// O5 (Eq. 4 line 3, the sum): acc_mn = sum_j a_mj * w_nj in int32.  Plain triple loop m, n, j.
//   a [M,K] int8, w [N,K] int8 (values in {-1,0,+1}; any int8 is accepted), acc [M,N] int32
void orc_contract(const int8_t* a, const int8_t* w, int M, int N, int K, int32_t* acc) {
#pragma omp parallel for schedule(static)
    for (long mn = 0; mn < (long)M * N; ++mn) {
        int m = (int)(mn / N), n = (int)(mn % N);
        const int8_t* ar = a + (long)m * K;
        const int8_t* wr = w + (long)n * K;
        int32_t s = 0;
        for (int j = 0; j < K; ++j) s += (int32_t)ar[j] * (int32_t)wr[j];
        acc[mn] = s;
    }
}

// O6 (Eq. 4 line 3, the scaling): s_m = alpha_m * beta_g ; y = (float)acc * s_m  (R6).
//   beta        [G] fp32, G >= 1 output groups of N/G consecutive channels each (R7; G=1 is the tensor scale)
//   y32         [M,N] fp32 or NULL
//   y64         [M,N] fp64 (double)acc*(double)alpha*(double)beta, the tolerance reference, or NULL
void orc_rescale(const int32_t* acc, const float* alpha, const float* beta, int G,
                 int M, int N, float* y32, double* y64) {
    int per = N / G;
    for (int m = 0; m < M; ++m)
        for (int n = 0; n < N; ++n) {
            float b = beta[n / per];
            long i = (long)m * N + n;
            if (y32) {
                float s = alpha[m] * b;
                y32[i] = (float)acc[i] * s;
            }
            if (y64) y64[i] = (double)acc[i] * (double)alpha[m] * (double)b;
        }
}

// The whole path, Eq. 4 top to bottom, from bf16 activations to fp32 / bf16 outputs.
// Any output pointer may be NULL except acc_out (scratch the caller owns).
void orc_ternary_linear(const uint16_t* x, const int8_t* w, const float* beta, int G,
                        int M, int N, int K,
                        int8_t* a_out, float* alpha_out, int32_t* acc_out,
                        float* y32_out, uint16_t* ybf16_out, double* y64_out) {
    orc_act_quant(x, M, K, a_out, alpha_out);
    orc_contract(a_out, w, M, N, K, acc_out);
    if (y32_out || y64_out) orc_rescale(acc_out, alpha_out, beta, G, M, N, y32_out, y64_out);
    if (ybf16_out) {
        for (int m = 0; m < M; ++m)
            for (int n = 0; n < N; ++n) {
                long i = (long)m * N + n;
                float s = alpha_out[m] * beta[n / (N / G)];
                ybf16_out[i] = f32_to_bf16_rne((float)acc_out[i] * s);
            }
    }
}

// O8: reference statement of "four two-bit codes per byte".  code = q + 1; value k of a row
// sits in byte k/4 at bits 2*(k%4).  The CUDA library's layout is private and different; this exists
// only so that tests can state the round-trip property on the CPU.  Returns the number of values
// outside {-1,0,1} (0 on success).
long orc_pack_ref(const int8_t* w, long n, uint8_t* packed) {
    long bad = 0;
    for (long i = 0; i < n / 4; ++i) {
        uint8_t b = 0;
        for (int c = 0; c < 4; ++c) {
            int q = w[4 * i + c];
            if (q < -1 || q > 1) { ++bad; q = 0; }
            b |= (uint8_t)((q + 1) << (2 * c));
        }
        packed[i] = b;
    }
    return bad;
}

void orc_unpack_ref(const uint8_t* packed, long n, int8_t* w) {
    for (long i = 0; i < n / 4; ++i)
        for (int c = 0; c < 4; ++c) w[4 * i + c] = (int8_t)(((packed[i] >> (2 * c)) & 3) - 1);
}

}  // extern "C"
