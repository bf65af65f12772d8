/*
 * oracle_mlp.c -- CPU oracle for the chained GEMM  A^l = act(A^{l-1} . W_l),  Y = A^L.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_2607_07862_b200/)
 * may include, link, import or execute this file; only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs do.  It shares no code with the
 * CUDA path.
 *
 * What it computes (the plain definition; the method reaches the same result faster
 * and approximates nothing):
 *   - "two-layer GEMM ... where the output of the first GEMM is directly consumed by
 *     the subsequent GEMM"                       PAPER.md:107 (section III-B)
 *   - "Y = XAB, X the input activation, A and B the weight matrices"
 *                                                  PAPER.md:161 (section IV)
 *   - "input and output data types are set to BF16, and the Tensor Core accumulator
 *     type is set to FP32"
 *   - the intermediate is a kernel OUTPUT written to memory (arrow (1)),
 *     hence every A^l is rounded to bf16 before the next layer reads it.
 *   - the activation comes from BASELINE.json configs, not from the paper (which omits
 *     it); reading c1/c2 of DESIGN.md: applied to the fp32 accumulator
 *     before the bf16 rounding, after every layer except the last.
 *
 * for l = 1..L, m in [0,M), n in [0,N_l):
 *     acc = 0.0f                                        (IEEE binary32)
 *     for k = 0 .. K_l-1 ascending:
 *         acc = acc + (float)A^{l-1}[m,k] * (float)W_l[k,n]
 *     if l < L: acc = act(acc)
 *     A^l[m,n] = bf16_rne(acc)
 *
 * The product of two bf16 values is exact in fp32 (8+8 significand bits <= 24), so
 * a*b+acc and fma(a,b,acc) are the same number; the build still passes
 * -ffp-contract=off and never -ffast-math.
 *
 * Loop nest: output columns n are independent, so they are split into blocks across
 * OpenMP threads and the two inner loops run k (ascending) then n-in-block.  Every
 * acc[m,n] still receives its K_l addends one by one in ascending k: the result does
 * not depend on the block width or on the thread count.  W_l is accepted in the
 * boundary layout [N_l x K_l] (K contiguous) and is first copied to a [K_l x N_l]
 * float array -- a layout change only.
 *
 * Pins (tests/test_oracle_pins.py): brute-force exact rational dot products on tiny
 * shapes, a hand-worked 2x3x2x2 example (tests/golden/), all-ones closed form, W=I
 * special cases, float64 library matmul within the analytic rounding bound, the int64
 * exactness certificate, row independence, power-of-two homogeneity, hidden-unit
 * permutation invariance, GeLU against torch's float64 tanh-GeLU, bf16 RNE ties and
 * torch's own fp32->bf16 cast.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORACLE_ACT_NONE = 0, ORACLE_ACT_RELU = 1, ORACLE_ACT_GELU_TANH = 2 };

/* bf16 -> fp32: the bf16 pattern is the top half of the binary32 pattern. */
float oracle_bf16_to_f32(uint16_t h) {
    uint32_t u = (uint32_t)h << 16;
    float f;
    memcpy(&f, &u, 4);
    return f;
}

/* fp32 -> bf16, IEEE round-to-nearest-even (reading c6).
 * Inputs are finite by construction; NaN is mapped to a quiet NaN so that the
 * poison tests can see it. */
uint16_t oracle_bf16_rne(float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x0040u);
    u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

/* tanh-form GeLU (reading c1), evaluated in double from the fp32
 * accumulator and returned as float:
 *   g(x) = 0.5 x (1 + tanh( sqrt(2/pi) (x + 0.044715 x^3) ))                */
float oracle_gelu_tanh(float x) {
    double xd = (double)x;
    double inner = 0.7978845608028654 * (xd + 0.044715 * xd * xd * xd);
    return (float)(0.5 * xd * (1.0 + tanh(inner)));
}

float oracle_act(float acc, int act) {
    switch (act) {
    case ORACLE_ACT_RELU: return acc > 0.0f ? acc : 0.0f; /* -0 and negatives -> +0 */
    case ORACLE_ACT_GELU_TANH: return oracle_gelu_tanh(acc);
    default: return acc;
    }
}

#define ORACLE_NB 64 /* output columns per block; any value gives the same bits */

/*
 * One layer.  A: [M x K] bf16 row-major.  W: [N x K] bf16, K contiguous.
 * out: [M x N] bf16 row-major.  acc_out (optional, may be NULL): the fp32
 * accumulators before activation, [M x N].
 * cert (optional, may be NULL): int64 exactness certificate for integer-valued
 * inputs (reading c7): cert[0] = max |partial sum| seen in int64,
 * cert[1] = number of (m,n) whose fp32 accumulator differs from the int64 sum,
 * cert[2] = 1 if some operand was not an integer.
 */
int oracle_gemm_layer(int M, int K, int N, const uint16_t *A, const uint16_t *W, int act,
                      uint16_t *out, float *acc_out, int64_t *cert, int threads) {
    if (M <= 0 || K <= 0 || N <= 0 || !A || !W || !out) return 1;
    float *Wt = (float *)malloc((size_t)K * N * sizeof(float));
    float *Af = (float *)malloc((size_t)M * K * sizeof(float));
    if (!Wt || !Af) { free(Wt); free(Af); return 4; }
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#endif
    /* layout change only: Wt[k][n] = (float) W[n][k] */
#pragma omp parallel for schedule(static)
    for (int k = 0; k < K; k++)
        for (int n = 0; n < N; n++) Wt[(size_t)k * N + n] = oracle_bf16_to_f32(W[(size_t)n * K + k]);
#pragma omp parallel for schedule(static)
    for (int m = 0; m < M; m++)
        for (int k = 0; k < K; k++) Af[(size_t)m * K + k] = oracle_bf16_to_f32(A[(size_t)m * K + k]);

    int64_t cert_max = 0, cert_bad = 0, cert_nonint = 0;
    int nblocks = (N + ORACLE_NB - 1) / ORACLE_NB;
#pragma omp parallel for schedule(dynamic, 1) reduction(max : cert_max) reduction(+ : cert_bad, cert_nonint)
    for (int b = 0; b < nblocks; b++) {
        int n0 = b * ORACLE_NB;
        int nw = N - n0 < ORACLE_NB ? N - n0 : ORACLE_NB;
        for (int m = 0; m < M; m++) {
            float acc[ORACLE_NB];
            for (int j = 0; j < nw; j++) acc[j] = 0.0f;
            const float *a = Af + (size_t)m * K;
            for (int k = 0; k < K; k++) { /* ascending k, one addend at a time */
                float x = a[k];
                const float *w = Wt + (size_t)k * N + n0;
                for (int j = 0; j < nw; j++) acc[j] = acc[j] + x * w[j];
            }
            if (cert) { /* the same sums in int64, beside the fp32 ones */
                for (int j = 0; j < nw; j++) {
                    int64_t s = 0, smax = 0;
                    for (int k = 0; k < K; k++) {
                        float x = a[k], y = Wt[(size_t)k * N + n0 + j];
                        if (x != (float)(int64_t)x || y != (float)(int64_t)y) cert_nonint = 1;
                        s += (int64_t)x * (int64_t)y;
                        int64_t as = s < 0 ? -s : s;
                        if (as > smax) smax = as;
                    }
                    if (smax > cert_max) cert_max = smax;
                    if ((double)acc[j] != (double)s) cert_bad += 1;
                }
            }
            for (int j = 0; j < nw; j++) {
                if (acc_out) acc_out[(size_t)m * N + n0 + j] = acc[j];
                out[(size_t)m * N + n0 + j] = oracle_bf16_rne(oracle_act(acc[j], act));
            }
        }
    }
    if (cert) { cert[0] = cert_max; cert[1] = cert_bad; cert[2] = cert_nonint; }
    free(Wt);
    free(Af);
    return 0;
}

/*
 * The chain.  widths[0..L]: K -> N_1 -> ... -> N_L.  W[l]: [widths[l+1] x widths[l]].
 * outs[l]: caller-allocated [M x widths[l+1]] bf16; outs[L-1] is Y, the others are
 * the hidden activations H_l.  act is applied after every layer except the last
 * (reading c2).  cert (optional): 3 int64 per layer.
 */
int oracle_mlp_chain(int M, int L, const int *widths, const uint16_t *X, const uint16_t *const *W,
                     int act, uint16_t *const *outs, int64_t *cert, int threads) {
    if (L <= 0 || !widths || !X || !W || !outs) return 1;
    const uint16_t *in = X;
    for (int l = 0; l < L; l++) {
        int rc = oracle_gemm_layer(M, widths[l], widths[l + 1], in, W[l], l < L - 1 ? act : ORACLE_ACT_NONE,
                                   outs[l], NULL, cert ? cert + 3 * l : NULL, threads);
        if (rc) return rc;
        in = outs[l];
    }
    return 0;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
