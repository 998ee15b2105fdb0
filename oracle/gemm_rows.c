/* ORACLE (test infrastructure, NOT the product): plain CPU definition of the two serving-phase
 * contractions, the decode GEMV and the prefill GEMM ("dense GEMM kernels" in
 * prefill, "GEMV-like operators" in decode; shapes from BASELINE.json configs 3-4).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code with the CUDA library.
 *
 * What it computes (SURVEY.md §8(a) a2/a3, §8(c) Oracle B), for every requested row i and every
 * column j, in ASCENDING k:
 *
 *     c64 += (double)A[i][k] * (double)W[k][j]          reference value
 *     s64 += fabs(that product)                         scale of the tolerance 1e-3 * sum|a*b|
 *     c32  = fmaf((float)A[i][k], (float)W[k][j], c32)  "computed in fp32 from bf16 inputs"
 *     y16  = bf16_rne(c32)                              the bf16 output of the definition
 *
 * bf16 operands are raw uint16 bit patterns; widening is exact (bits << 16).  bf16 x bf16 products
 * are exact in fp32 and in double, so only the additions round.
 *
 * Logical shapes A[m][k], W[k][n].  Physical W layout:
 *     w_layout 0 (NK): W_phys[j*ldw + k]   (K contiguous, nn.Linear storage)
 *     w_layout 1 (KN): W_phys[k*ldw + j]   (N contiguous, "[3584 x 18944]" as written)
 *
 * Pins (tests/test_oracle_gemm.py): identity / permutation / ones matrices (exact), exact-rational
 * brute force on tiny shapes, numpy float64 matmul of the widened inputs, bf16 rounding against
 * ties and against torch's conversion, |c32 - c64| <= K 2^-24 s64.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

static inline float bf16_to_f32(uint16_t h)
{
    uint32_t u = (uint32_t)h << 16;
    float f;
    memcpy(&f, &u, 4);
    return f;
}

/* fp32 -> bf16, round to nearest, ties to even.  NaN is kept quiet. */
uint16_t oracle_f32_to_bf16_rne(float f)
{
    uint32_t u;
    memcpy(&u, &f, 4);
    if ((u & 0x7FFFFFFFu) > 0x7F800000u)
        return (uint16_t)((u >> 16) | 0x0040u);
    uint32_t lsb = (u >> 16) & 1u;
    u += 0x7FFFu + lsb;
    return (uint16_t)(u >> 16);
}

float oracle_bf16_to_f32(uint16_t h) { return bf16_to_f32(h); }

/* rows[r] selects the A row; outputs are [nrows][n] row-major.  Any output pointer may be NULL. */
void oracle_gemm_rows(const uint16_t *a, long long lda, const uint16_t *w, long long ldw, int w_layout,
                      int n, int k, const int *rows, int nrows,
                      double *c64, double *s64, float *c32, uint16_t *y16)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int r = 0; r < nrows; ++r) {
        for (int j = 0; j < n; ++j) {
            const uint16_t *arow = a + (long long)rows[r] * lda;
            double acc64 = 0.0, sum_abs = 0.0;
            float acc32 = 0.0f;
            for (int kk = 0; kk < k; ++kk) {
                uint16_t wb = (w_layout == 0) ? w[(long long)j * ldw + kk] : w[(long long)kk * ldw + j];
                float af = bf16_to_f32(arow[kk]);
                float wf = bf16_to_f32(wb);
                double p = (double)af * (double)wf;
                acc64 += p;
                sum_abs += fabs(p);
                acc32 = fmaf(af, wf, acc32);
            }
            long long o = (long long)r * n + j;
            if (c64) c64[o] = acc64;
            if (s64) s64[o] = sum_abs;
            if (c32) c32[o] = acc32;
            if (y16) y16[o] = oracle_f32_to_bf16_rne(acc32);
        }
    }
}
