/*
 * ORACLE, third form (test infrastructure only; same rules as csg_oracle.c): 2D orders FROM COORDINATES.
 *
 * It exists to give the whole interval-abundance histogram of BASELINE.json configs[4] (N = 262144, all
 * 262143 bins) in minutes and by a route that shares nothing with the relation matrix: no bitset, no AND,
 * no popcount, no element indices (pin P6).
 *
 * Definition it writes out.  In a random 2D order (2D Minkowski diamond in light-cone coordinates, DESIGN.md
 * reading A17) element a precedes element b iff u_a < u_b and v_a < v_b (both strict).  The interval between
 * a related pair is the set of elements that follow a and precede b (Sec. 4.1: "the number of
 * elements k both to the future of element i and to the past of element j"), i.e. the sprinkled points
 * strictly inside the rectangle (u_a, u_b) x (v_a, v_b):
 *
 *      n_ab = #{ c : u_a < u_c < u_b  and  v_a < v_c < v_b },      counts[n_ab] += 1 for every related pair.
 *
 * Method (plain dominance counting): sort the points by u; replace v by its rank.  For each lower element a,
 * walk the later points b in increasing u and keep a Fenwick (binary indexed) tree over the v-ranks of the
 * points met so far whose v exceeds v_a.  When b itself has v_b > v_a it is related to a and n_ab is the number
 * of stored ranks below rank(v_b) -- every stored point c has u_a < u_c < u_b (met after a, before b) and
 * v_a < v_c, and the prefix sum adds v_c < v_b.  O(N^2 log N) in all, OpenMP over a, thread-private
 * histograms.
 *
 * Equal coordinates would make "strictly inside" differ from a comparison of ranks, so the function refuses
 * them (returns -1): the seeded configs have none.
 *
 * Pins (tests/test_oracle_pins.py): equal, bin for bin, to the triple loop csg_oracle_counts on the generator's
 * relation matrix of the same coordinates (N <= 3000 and configs[0]); to Algorithm 5 at configs[1]; to a
 * brute-force O(N^3) count from the coordinates; sum = C(N,2) - inversions.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    double key;
    int64_t id;
} keyed_t;

static int cmp_keyed(const void *a, const void *b)
{
    const keyed_t *x = (const keyed_t *)a, *y = (const keyed_t *)b;
    if (x->key < y->key) return -1;
    if (x->key > y->key) return 1;
    return 0;
}

/* coords: N rows of (u, v), any order.  counts[0..kmax] overwritten.  Only related pairs whose LOWER element is
 * one of the rows id_begin <= id < id_end of `coords` are counted (0, N for all of them): the same split by first
 * element as csg_alg5_counts_rows, so that a partial Algorithm-5 run can be checked block by block.
 * Returns 0, -1 if two points share a u or a v value, -2 if out of memory. */
int csg_dominance2d_counts_rows(const double *coords, int64_t N, int64_t kmax, int64_t id_begin, int64_t id_end,
                                int64_t *counts)
{
    const int64_t nb = kmax + 1;
    memset(counts, 0, (size_t)nb * sizeof(int64_t));
    if (N < 2)
        return 0;
    keyed_t *byu = (keyed_t *)malloc((size_t)N * sizeof(keyed_t));
    keyed_t *byv = (keyed_t *)malloc((size_t)N * sizeof(keyed_t));
    int32_t *vrank_of_id = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int32_t *vr = (int32_t *)malloc((size_t)N * sizeof(int32_t)); /* v-rank (1-based) of the a-th point in u order */
    uint8_t *wanted = (uint8_t *)malloc((size_t)N);              /* is the a-th point in u order a wanted lower element? */
    if (!byu || !byv || !vrank_of_id || !vr || !wanted) {
        free(byu); free(byv); free(vrank_of_id); free(vr); free(wanted);
        return -2;
    }
    for (int64_t n = 0; n < N; ++n) {
        byu[n].key = coords[2 * n];
        byu[n].id = n;
        byv[n].key = coords[2 * n + 1];
        byv[n].id = n;
    }
    qsort(byu, (size_t)N, sizeof(keyed_t), cmp_keyed);
    qsort(byv, (size_t)N, sizeof(keyed_t), cmp_keyed);
    int ties = 0;
    for (int64_t n = 1; n < N; ++n)
        if (byu[n].key == byu[n - 1].key || byv[n].key == byv[n - 1].key)
            ties = 1;
    for (int64_t n = 0; n < N; ++n)
        vrank_of_id[byv[n].id] = (int32_t)(n + 1);
    for (int64_t a = 0; a < N; ++a) {
        vr[a] = vrank_of_id[byu[a].id];
        wanted[a] = (uint8_t)(byu[a].id >= id_begin && byu[a].id < id_end);
    }
    free(byu); free(byv); free(vrank_of_id);
    if (ties) {
        free(vr); free(wanted);
        return -1;
    }
    int oom = 0;
#pragma omp parallel
    {
        int64_t *priv = (int64_t *)calloc((size_t)nb, sizeof(int64_t));
        int32_t *tree = (int32_t *)malloc((size_t)(N + 1) * sizeof(int32_t)); /* Fenwick tree over ranks 1..N */
        if (!priv || !tree) {
#pragma omp atomic write
            oom = 1;
        }
#pragma omp for schedule(dynamic, 16)
        for (int64_t a = 0; a < N; ++a) {
            if (!priv || !tree || !wanted[a])
                continue;
            memset(tree, 0, (size_t)(N + 1) * sizeof(int32_t));
            const int32_t va = vr[a];
            for (int64_t b = a + 1; b < N; ++b) {
                const int32_t vb = vr[b];
                if (vb < va)
                    continue; /* not related to a, and never inside a rectangle that starts at a */
                int64_t n = 0; /* stored ranks < vb */
                for (int32_t x = vb - 1; x > 0; x -= x & (-x))
                    n += tree[x];
                if (n <= kmax)
                    priv[n] += 1;
                for (int32_t x = vb; x <= N; x += x & (-x))
                    tree[x] += 1;
            }
        }
#pragma omp critical
        if (priv)
            for (int64_t n = 0; n < nb; ++n)
                counts[n] += priv[n];
        free(priv);
        free(tree);
    }
    free(vr);
    free(wanted);
    return oom ? -2 : 0;
}

int csg_dominance2d_counts(const double *coords, int64_t N, int64_t kmax, int64_t *counts)
{
    return csg_dominance2d_counts_rows(coords, N, kmax, 0, N, counts);
}

/* P5: number of related pairs of a 2D order = C(N,2) - inversions of the v-ranks read in u order (a pair is
 * related iff it is NOT an inversion); by merge sort, O(N log N).  Returns -1 on ties, -2 out of memory. */
static int64_t merge_count(int32_t *x, int32_t *tmp, int64_t lo, int64_t hi)
{
    if (hi - lo < 2)
        return 0;
    const int64_t mid = lo + (hi - lo) / 2;
    int64_t inv = merge_count(x, tmp, lo, mid) + merge_count(x, tmp, mid, hi);
    int64_t p = lo, q = mid, o = lo;
    while (p < mid && q < hi) {
        if (x[q] < x[p]) {
            inv += mid - p; /* x[q] jumps over everything left in the first half */
            tmp[o++] = x[q++];
        } else {
            tmp[o++] = x[p++];
        }
    }
    while (p < mid) tmp[o++] = x[p++];
    while (q < hi) tmp[o++] = x[q++];
    memcpy(x + lo, tmp + lo, (size_t)(hi - lo) * sizeof(int32_t));
    return inv;
}

int64_t csg_dominance2d_relations(const double *coords, int64_t N)
{
    if (N < 2)
        return 0;
    keyed_t *byu = (keyed_t *)malloc((size_t)N * sizeof(keyed_t));
    keyed_t *byv = (keyed_t *)malloc((size_t)N * sizeof(keyed_t));
    int32_t *vrank_of_id = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int32_t *vr = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int32_t *tmp = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    if (!byu || !byv || !vrank_of_id || !vr || !tmp) {
        free(byu); free(byv); free(vrank_of_id); free(vr); free(tmp);
        return -2;
    }
    for (int64_t n = 0; n < N; ++n) {
        byu[n].key = coords[2 * n];
        byu[n].id = n;
        byv[n].key = coords[2 * n + 1];
        byv[n].id = n;
    }
    qsort(byu, (size_t)N, sizeof(keyed_t), cmp_keyed);
    qsort(byv, (size_t)N, sizeof(keyed_t), cmp_keyed);
    int ties = 0;
    for (int64_t n = 1; n < N; ++n)
        if (byu[n].key == byu[n - 1].key || byv[n].key == byv[n - 1].key)
            ties = 1;
    for (int64_t n = 0; n < N; ++n)
        vrank_of_id[byv[n].id] = (int32_t)(n + 1);
    for (int64_t a = 0; a < N; ++a)
        vr[a] = vrank_of_id[byu[a].id];
    const int64_t inv = merge_count(vr, tmp, 0, N);
    free(byu); free(byv); free(vrank_of_id); free(vr); free(tmp);
    if (ties)
        return -1;
    return N * (N - 1) / 2 - inv;
}
