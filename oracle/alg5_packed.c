/*
 * ORACLE, second form (test infrastructure only; same rules as csg_oracle.c).
 *
 * Algorithm 5 "Optimized Cardinality Measurement" of the paper restated step by step in plain C
 * (Sec. 4.3): loop over the N(N-1)/2 pairs (OpenMP), `continue`
 * when the pair is unrelated (l.4-5), m = partial vector product of rows i and j (l.7; AND + popcount
 * over the blocks covering columns i..j with masks on the two end blocks),
 * then c[m]++ in a thread-private array that is reduced at the end.
 * Readings A2 (no reserved slot 0) and A3 (open range i<k<j) as in csg_oracle.c.
 *
 * It exists because the plain triple loop cannot finish at N >= 65536.  Pin (P13): it must equal
 * csg_oracle_counts bit for bit wherever both run (tests/test_oracle_pins.py); it shares no code with
 * the CUDA path.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* popcount of (a & b) restricted to bit columns lo..hi inclusive (partial_vecprod). */
static int64_t partial_vecprod(const uint64_t *a, const uint64_t *b, int64_t lo, int64_t hi)
{
    if (lo > hi)
        return 0;
    int64_t wlo = lo >> 6, whi = hi >> 6;
    uint64_t mlo = ~0ULL << (lo & 63);
    uint64_t mhi = ((hi & 63) == 63) ? ~0ULL : ((1ULL << ((hi & 63) + 1)) - 1ULL);
    if (wlo == whi)
        return __builtin_popcountll(a[wlo] & b[wlo] & mlo & mhi);
    int64_t m = __builtin_popcountll(a[wlo] & b[wlo] & mlo);
    for (int64_t w = wlo + 1; w < whi; ++w)
        m += __builtin_popcountll(a[w] & b[w]);
    m += __builtin_popcountll(a[whi] & b[whi] & mhi);
    return m;
}

int csg_alg5_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Rows i in [row_begin, row_end) only (row_begin=0,row_end=N for the whole set): lets bench.py time a
 * bounded sample of the workload.  tests_done (may be NULL) receives sum over ALL pairs i<j visited,
 * related or not, of (j-i-1) = the ordered-triple tests those rows stand for. */
void csg_alg5_counts_rows(const uint64_t *bits, int64_t N, int64_t stride_words, int64_t kmax,
                          int64_t row_begin, int64_t row_end, int64_t *counts, int64_t *tests_done)
{
    int64_t nb = kmax + 1;
    memset(counts, 0, (size_t)nb * sizeof(int64_t));
    int64_t tests = 0;
#pragma omp parallel reduction(+ : tests)
    {
        int64_t *priv = (int64_t *)calloc((size_t)nb, sizeof(int64_t));
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = row_begin; i < row_end; ++i) {
            const uint64_t *ri = bits + i * stride_words;
            for (int64_t j = i + 1; j < N; ++j) {
                tests += j - i - 1;
                if (!((ri[j >> 6] >> (j & 63)) & 1ULL))
                    continue;
                int64_t m = partial_vecprod(ri, bits + j * stride_words, i + 1, j - 1);
                if (m <= kmax)
                    priv[m] += 1;
            }
        }
#pragma omp critical
        for (int64_t n = 0; n < nb; ++n)
            counts[n] += priv[n];
        free(priv);
    }
    if (tests_done)
        *tests_done = tests;
}

void csg_alg5_counts(const uint64_t *bits, int64_t N, int64_t stride_words, int64_t kmax, int64_t *counts)
{
    csg_alg5_counts_rows(bits, N, stride_words, kmax, 0, N, counts, NULL);
}
