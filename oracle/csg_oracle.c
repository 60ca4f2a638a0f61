/*
 * ORACLE (test infrastructure only -- never linked into or imported by the product path).
 *
 * Plain, single-threaded, obviously-correct C restatement of what the hot path computes:
 * the interval-abundance histogram of a causal set and the Benincasa-Dowker action built from it.
 * It shares no code, header, table or helper with paper_1709_03013_b200/ (the CUDA path).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Source of every definition: /root/reference/PAPER.md (arXiv:1709.03013), cited per function as
 * PAPER.md:<line> + section/equation.  Readings of silent/ambiguous passages are listed in DESIGN.md
 * ("Readings") under the A-numbers quoted here.
 *
 * Parity pins (tests/test_oracle_pins.py): matrix-square identity, hand posets with closed forms,
 * exhaustive N! 2D orders with exact rational expectations, 2D dominance counting from coordinates,
 * Eq.5 in exact rational arithmetic, Eq.5(eps=1)==Eq.4.  Nothing here is "parity unpinned".
 */
#include <stdint.h>
#include <stddef.h>
#include <math.h>

/* Relation-matrix layout (Sec. 3.1-3.2: rows of 64-bit blocks, padding bits zero;
 * LSB-first within a block per get_bitmask=(1<<offset)-1).  Bit c of row r is
 * bit (c%64) of word bits[r*stride_words + c/64]. */
static int get_bit(const uint64_t *bits, int64_t stride_words, int64_t r, int64_t c)
{
    return (int)((bits[r * stride_words + (c >> 6)] >> (c & 63)) & 1u);
}

/* Expand the packed matrix to one byte per entry: B[r*N + c] in {0,1}.  (the oracle works
 * on a byte matrix expanded from the SAME packed bitset the GPU gets.) */
void csg_oracle_expand(const uint64_t *bits, int64_t N, int64_t stride_words, uint8_t *B)
{
    for (int64_t r = 0; r < N; ++r)
        for (int64_t c = 0; c < N; ++c)
            B[r * N + c] = (uint8_t)get_bit(bits, stride_words, r, c);
}

/* Naive action algorithm, PAPER.md:395 (Sec. 4.1): "three nested for loops ... For each non-zero entry
 * (i, j) of the causal matrix, with i < j due to time-ordering, we calculate the number of elements k both
 * [to] the future of element i and to the past of element j and then add one to the array of interval
 * abundances at index k."  Fig. 2 caption: inner product of rows i and j between columns
 * i and j.  Reading A3: the open range i<k<j.  Reading A1/A2: counts[n] is 0-based (= paper's n_{n+1}).
 * Reading A10: unrelated pairs contribute nothing.  Pairs with n > kmax are not counted anywhere.
 * counts has kmax+1 entries and is overwritten. */
void csg_oracle_counts(const uint8_t *B, int64_t N, int64_t kmax, int64_t *counts)
{
    for (int64_t n = 0; n <= kmax; ++n)
        counts[n] = 0;
    for (int64_t i = 0; i < N; ++i) {
        for (int64_t j = i + 1; j < N; ++j) {
            if (!B[i * N + j])
                continue;
            int64_t n = 0;
            for (int64_t k = i + 1; k < j; ++k)
                n += (int64_t)(B[i * N + k] & B[j * N + k]);
            if (n <= kmax)
                counts[n] += 1;
        }
    }
}

/* Interval size of ONE pair straight from the packed matrix, bit by bit (no popcount, no word tricks);
 * used for sampled checks at sizes where the N*N byte matrix does not fit.
 * Returns -1 if i>=j or the pair is unrelated.  PAPER.md:395, 59. */
int64_t csg_oracle_pair(const uint64_t *bits, int64_t N, int64_t stride_words, int64_t i, int64_t j)
{
    if (i < 0 || j >= N || i >= j)
        return -1;
    if (!get_bit(bits, stride_words, i, j))
        return -1;
    int64_t n = 0;
    for (int64_t k = i + 1; k < j; ++k)
        n += get_bit(bits, stride_words, i, k) & get_bit(bits, stride_words, j, k);
    return n;
}

/* Local (non-smeared) action.
 * dim==2: Eq. (4): S = 2(N - 2 n_1 + 4 n_2 - 2 n_3), with n_i = counts[i-1] (A1).
 * dim==4: NOT IN PAPER (reading A8): standard Benincasa-Dowker d=4 form
 *         S = (4/sqrt 6) (N - N_0 + 9 N_1 - 16 N_2 + 8 N_3), integer combination first, one scale last.
 * Returns NaN for any other dim. */
double csg_oracle_action_local(int dim, int64_t N, const int64_t *counts)
{
    if (dim == 2) {
        int64_t I2 = N - 2 * counts[0] + 4 * counts[1] - 2 * counts[2];
        return 2.0 * (double)I2;
    }
    if (dim == 4) {
        int64_t I4 = N - counts[0] + 9 * counts[1] - 16 * counts[2] + 8 * counts[3];
        return (4.0 / sqrt(6.0)) * (double)I4;
    }
    return NAN;
}

/* Smearing weight, Eq. (5):
 *   f_2(i,e) = (1-e)^i [ 1 - 2 e i/(1-e) + e^2 i(i-1) / (2 (1-e)^2) ]
 * written with the bracket multiplied out (reading A7) so that e -> 1 needs no 0/0:
 *   f_2(i,e) = (1-e)^i - 2 e i (1-e)^(i-1) + (e^2 i(i-1)/2) (1-e)^(i-2). */
double csg_oracle_f2(int64_t i, double e)
{
    double x = 1.0 - e;
    double di = (double)i;
    double t0 = pow(x, di);
    double t1 = (i >= 1) ? 2.0 * e * di * pow(x, di - 1.0) : 0.0;
    double t2 = (i >= 2) ? 0.5 * e * e * di * (di - 1.0) * pow(x, di - 2.0) : 0.0;
    return t0 - t1 + t2;
}

/* Smeared action in 1+1 dimensions, Eq. (5):
 *   S_e = 2 e [ N - 2 e sum_{i=1}^{N-1} n_i f_2(i-1, e) ]  =  2 e [ N - 2 e sum_{k=0}^{kmax} counts[k] f_2(k,e) ]
 * (A1: n_i = counts[i-1]; A6: k runs 0..N-2; the caller passes kmax = N-2 for the exact sum).
 * Reading A14: ascending k, Kahan-compensated double sum.  If abs_scale != NULL it receives
 * 4 e^2 sum_k |counts[k] f_2(k,e)|, the scale against which tests set the tolerance. */
double csg_oracle_action_smeared_2d(int64_t N, int64_t kmax, const int64_t *counts, double e, double *abs_scale)
{
    double sum = 0.0, comp = 0.0, asum = 0.0;
    for (int64_t k = 0; k <= kmax; ++k) {
        double term = (double)counts[k] * csg_oracle_f2(k, e);
        double y = term - comp;
        double t = sum + y;
        comp = (t - sum) - y;
        sum = t;
        asum += fabs(term);
    }
    if (abs_scale)
        *abs_scale = 4.0 * e * e * asum;
    return 2.0 * e * ((double)N - 2.0 * e * sum);
}

/* Smeared action in 3+1 dimensions.  NOT IN PAPER (it cites [5],[19],[24] for other dimensions);
 * DESIGN.md reading A9: the d=4 member of the same family,
 *   S_e = (4/sqrt 6) sqrt(e) [ N - e sum_k counts[k] f_4(k,e) ],
 *   f_4(k,e) = (1-e)^k [ 1 - 9 e k/(1-e) + 8 e^2 k(k-1)/(1-e)^2 - (4/3) e^3 k(k-1)(k-2)/(1-e)^3 ],
 * bracket multiplied out as for f_2 so that e -> 1 gives the local weights 1, -9, 16, -8 (reading A8).
 * "Parity unpinned" against the paper (nothing printed there); pinned against exact rational evaluation of this
 * formula and against its e = 1 limit. */
double csg_oracle_f4(int64_t i, double e)
{
    double x = 1.0 - e;
    double di = (double)i;
    double t0 = pow(x, di);
    double t1 = (i >= 1) ? 9.0 * e * di * pow(x, di - 1.0) : 0.0;
    double t2 = (i >= 2) ? 8.0 * e * e * di * (di - 1.0) * pow(x, di - 2.0) : 0.0;
    double t3 = (i >= 3) ? (4.0 / 3.0) * e * e * e * di * (di - 1.0) * (di - 2.0) * pow(x, di - 3.0) : 0.0;
    return ((t0 - t1) + t2) - t3;
}

double csg_oracle_action_smeared_4d(int64_t N, int64_t kmax, const int64_t *counts, double e, double *abs_scale)
{
    double sum = 0.0, comp = 0.0, asum = 0.0;
    for (int64_t k = 0; k <= kmax; ++k) {
        double term = (double)counts[k] * csg_oracle_f4(k, e);
        double y = term - comp;
        double t = sum + y;
        comp = (t - sum) - y;
        sum = t;
        asum += fabs(term);
    }
    double pref = (4.0 / sqrt(6.0)) * sqrt(e);
    if (abs_scale)
        *abs_scale = pref * e * asum;
    return pref * ((double)N - e * sum);
}
