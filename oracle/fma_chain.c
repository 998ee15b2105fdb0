/* ORACLE (test infrastructure, NOT the product): plain CPU definition of the A.I.-parameterised
 * FMA-chain roofline kernel.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code with the CUDA library.
 *
 * What it computes (SURVEY.md §8(a) a1 / §8(c) Oracle A; BASELINE.json north_star, configs 1-2;
 * the paper only says "a synthetic roofline kernel" swept over A.I.):
 *
 *     for every element i:   y <- in[i];   repeat k times:  y <- fmaf(a, y, b);   out[i] <- y
 *
 * fp32, IEEE round-to-nearest-even, FUSED (one rounding per step), steps in this order.
 * Per element: 4 B read + 4 B written, 2k FLOP, so A.I. = 2k/8 FLOP/B (BASELINE.json config 1).
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off (no -ffast-math, no FTZ/DAZ).  fmaf() is the C99
 * libm function: exact a*y+b rounded once.  OpenMP only splits the independent elements.
 *
 * Pins (tests/test_oracle_fma.py): exact-rational emulation of the fused step, closed form
 * y_k = 1 + a^k (y0 - 1) within 2^-15 (1 - a^k), fixed point y0 = 1, exact k = 1 cases,
 * composition chain_{k1+k2} = chain_{k2} o chain_{k1}, monotonicity and range.
 */
#include <math.h>
#include <stddef.h>

void oracle_fma_chain(const float *in, float *out, size_t n, unsigned k, float a, float b)
{
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; ++i) {
        float y = in[i];
        for (unsigned s = 0; s < k; ++s)
            y = fmaf(a, y, b);
        out[i] = y;
    }
}

/* Number of 32-bit patterns that differ between two float arrays (bit compare, not value compare). */
size_t oracle_count_bit_mismatches(const float *x, const float *y, size_t n, long long *first)
{
    size_t bad = 0;
    long long f = -1;
    const unsigned *ux = (const unsigned *)x, *uy = (const unsigned *)y;
    for (size_t i = 0; i < n; ++i)
        if (ux[i] != uy[i]) {
            if (f < 0) f = (long long)i;
            ++bad;
        }
    if (first) *first = f;
    return bad;
}
