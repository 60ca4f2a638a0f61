/*
 * Seeded synthetic INPUT generator (shared by the oracle side and the CUDA side; holds none of the
 * method's arithmetic: no interval counting, no histogram, no action).
 *
 * It stands in for the paper's coordinate generation + linking (Sec. 2) on the flat
 * causal diamonds that BASELINE.json's configs name; recipe = DESIGN.md "Input recipe" (reading A17).
 *   - RNG: splitmix64 used as a counter-based generator, value n = mix(seed + (n+1)*GOLDEN),
 *     uniform double in [0,1) = (x >> 11) * 2^-53.
 *   - 2D: light-cone coordinates u,v i.i.d. uniform[0,1); i<j related iff u_i<u_j and v_i<v_j (strict);
 *     elements sorted by (u+v, u, draw index).
 *   - 4D: rejection sampling of (t,x,y,z), t in [0,1), x,y,z in [-1/2,1/2), accept iff
 *     x^2+y^2+z^2 < min(t,1-t)^2 (Alexandrov interval of height 1); related iff dt>0 and
 *     dt*dt > dx*dx+dy*dy+dz*dz (strict, doubles, no sqrt); sorted by (t, draw index).
 *   - (1+1) de Sitter slab, the paper's own workload: eta = atan(tan(eta0) (2a-1)) with a
 *     uniform (inverse CDF of rho(eta|eta0) = sec^2 eta / tan eta0 ... normalised on [-eta0, eta0]), theta =
 *     2 pi b; related iff pi - |pi - |dtheta|| < |deta|; sorted by (eta, draw index).
 *   - Output: symmetric packed matrix, zero diagonal, zero padding, LSB-first 64-bit words,
 *     row stride = 4*ceil(N/256) words (rows 256-bit aligned as PAPER.md:169).
 * Compile without -ffast-math / FMA contraction (-ffp-contract=off) so comparisons are reproducible.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define GOLDEN 0x9E3779B97F4A7C15ULL

static uint64_t mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static double uniform01(uint64_t seed, uint64_t n)
{
    uint64_t x = mix64(seed + (n + 1ULL) * GOLDEN);
    return (double)(x >> 11) * (1.0 / 9007199254740992.0);
}

int64_t csg_gen_stride_words(int64_t N) { return 4 * ((N + 255) / 256); }

typedef struct { double key, key2; int64_t idx; } sort_item;
static int cmp_item(const void *a, const void *b)
{
    const sort_item *x = (const sort_item *)a, *y = (const sort_item *)b;
    if (x->key < y->key) return -1;
    if (x->key > y->key) return 1;
    if (x->key2 < y->key2) return -1;
    if (x->key2 > y->key2) return 1;
    return (x->idx > y->idx) - (x->idx < y->idx);
}

/* coords: N x 2 doubles (u,v), written in sorted (time) order. */
int csg_gen_coords_2d(uint64_t seed, int64_t N, double *coords)
{
    sort_item *it = (sort_item *)malloc((size_t)(N > 0 ? N : 1) * sizeof(sort_item));
    double *raw = (double *)malloc((size_t)(N > 0 ? N : 1) * 2 * sizeof(double));
    if (!it || !raw) { free(it); free(raw); return -1; }
    for (int64_t n = 0; n < N; ++n) {
        double u = uniform01(seed, 2 * (uint64_t)n), v = uniform01(seed, 2 * (uint64_t)n + 1);
        raw[2 * n] = u; raw[2 * n + 1] = v;
        it[n].key = u + v; it[n].key2 = u; it[n].idx = n;
    }
    qsort(it, (size_t)N, sizeof(sort_item), cmp_item);
    for (int64_t n = 0; n < N; ++n) {
        coords[2 * n] = raw[2 * it[n].idx];
        coords[2 * n + 1] = raw[2 * it[n].idx + 1];
    }
    free(it); free(raw);
    return 0;
}

/* coords: N x 4 doubles (t,x,y,z), written in sorted (time) order. */
int csg_gen_coords_4d(uint64_t seed, int64_t N, double *coords)
{
    sort_item *it = (sort_item *)malloc((size_t)(N > 0 ? N : 1) * sizeof(sort_item));
    double *raw = (double *)malloc((size_t)(N > 0 ? N : 1) * 4 * sizeof(double));
    if (!it || !raw) { free(it); free(raw); return -1; }
    uint64_t attempt = 0;
    for (int64_t n = 0; n < N;) {
        double t = uniform01(seed, 4 * attempt);
        double x = uniform01(seed, 4 * attempt + 1) - 0.5;
        double y = uniform01(seed, 4 * attempt + 2) - 0.5;
        double z = uniform01(seed, 4 * attempt + 3) - 0.5;
        ++attempt;
        double h = (t < 1.0 - t) ? t : 1.0 - t;
        if (x * x + y * y + z * z < h * h) {
            raw[4 * n] = t; raw[4 * n + 1] = x; raw[4 * n + 2] = y; raw[4 * n + 3] = z;
            it[n].key = t; it[n].key2 = 0.0; it[n].idx = n;
            ++n;
        }
    }
    qsort(it, (size_t)N, sizeof(sort_item), cmp_item);
    for (int64_t n = 0; n < N; ++n)
        memcpy(coords + 4 * n, raw + 4 * it[n].idx, 4 * sizeof(double));
    free(it); free(raw);
    return 0;
}

/* coords: N x 2 doubles (eta, theta), written in sorted (conformal time) order. */
int csg_gen_coords_ds2(uint64_t seed, int64_t N, double eta0, double *coords)
{
    sort_item *it = (sort_item *)malloc((size_t)(N > 0 ? N : 1) * sizeof(sort_item));
    double *raw = (double *)malloc((size_t)(N > 0 ? N : 1) * 2 * sizeof(double));
    if (!it || !raw) { free(it); free(raw); return -1; }
    const double T = tan(eta0);
    for (int64_t n = 0; n < N; ++n) {
        double a = uniform01(seed, 2 * (uint64_t)n), b = uniform01(seed, 2 * (uint64_t)n + 1);
        raw[2 * n] = atan(T * (2.0 * a - 1.0));
        raw[2 * n + 1] = 6.28318530717958647692 * b;
        it[n].key = raw[2 * n]; it[n].key2 = 0.0; it[n].idx = n;
    }
    qsort(it, (size_t)N, sizeof(sort_item), cmp_item);
    for (int64_t n = 0; n < N; ++n) {
        coords[2 * n] = raw[2 * it[n].idx];
        coords[2 * n + 1] = raw[2 * it[n].idx + 1];
    }
    free(it); free(raw);
    return 0;
}

/* In-place transpose of a 64x64 bit block held as 64 words (row r = a[r], column c = bit c). */
static void transpose64(uint64_t a[64])
{
    uint64_t m = 0x00000000FFFFFFFFULL;
    for (int j = 32; j != 0; j >>= 1, m ^= (m << j)) {
        for (int k = 0; k < 64; k = (k + j + 1) & ~j) {
            uint64_t t = ((a[k] >> j) ^ a[k + j]) & m;
            a[k] ^= t << j;
            a[k + j] ^= t;
        }
    }
}

/* Fill the strictly-upper triangle row by row (thread-safe: row i only writes row i), then mirror it
 * into the lower triangle with 64x64 block transposes.  bits must hold N*stride zero-initialised words. */
static void mirror_lower(uint64_t *bits, int64_t N, int64_t stride)
{
    int64_t nb = (N + 63) / 64;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t bj = 0; bj < nb; ++bj) {           /* destination block-row */
        uint64_t blk[64];
        for (int64_t bi = 0; bi <= bj; ++bi) {      /* source block-row (upper: rows bi, cols bj) */
            for (int r = 0; r < 64; ++r) {
                int64_t row = bi * 64 + r;
                blk[r] = (row < N) ? bits[row * stride + bj] : 0ULL;
            }
            if (bi == bj) {                          /* diagonal block: keep its upper part too */
                uint64_t up[64];
                memcpy(up, blk, sizeof(up));
                transpose64(blk);
                for (int r = 0; r < 64; ++r) {
                    int64_t row = bj * 64 + r;
                    if (row < N) bits[row * stride + bi] = up[r] | blk[r];
                }
            } else {
                transpose64(blk);
                for (int r = 0; r < 64; ++r) {
                    int64_t row = bj * 64 + r;
                    if (row < N) bits[row * stride + bi] = blk[r];
                }
            }
        }
    }
}

int csg_gen_relations_2d(const double *coords, int64_t N, uint64_t *bits)
{
    int64_t stride = csg_gen_stride_words(N);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) {
        double ui = coords[2 * i], vi = coords[2 * i + 1];
        uint64_t *row = bits + i * stride;
        for (int64_t j = i + 1; j < N; ++j) {
            if (ui < coords[2 * j] && vi < coords[2 * j + 1])
                row[j >> 6] |= 1ULL << (j & 63);
        }
    }
    mirror_lower(bits, N, stride);
    return 0;
}

int csg_gen_relations_4d(const double *coords, int64_t N, uint64_t *bits)
{
    int64_t stride = csg_gen_stride_words(N);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) {
        const double *ci = coords + 4 * i;
        uint64_t *row = bits + i * stride;
        for (int64_t j = i + 1; j < N; ++j) {
            const double *cj = coords + 4 * j;
            double dt = cj[0] - ci[0], dx = cj[1] - ci[1], dy = cj[2] - ci[2], dz = cj[3] - ci[3];
            double s2 = dx * dx + dy * dy;
            s2 = s2 + dz * dz;
            if (dt > 0.0 && dt * dt > s2)
                row[j >> 6] |= 1ULL << (j & 63);
        }
    }
    mirror_lower(bits, N, stride);
    return 0;
}

int csg_gen_relations_ds2(const double *coords, int64_t N, uint64_t *bits)
{
    int64_t stride = csg_gen_stride_words(N);
    const double PI = 3.14159265358979323846;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) {
        double ei = coords[2 * i], ti = coords[2 * i + 1];
        uint64_t *row = bits + i * stride;
        for (int64_t j = i + 1; j < N; ++j) {
            double dth = fabs(ti - coords[2 * j + 1]);
            double lhs = PI - fabs(PI - dth);
            if (lhs < fabs(ei - coords[2 * j]))
                row[j >> 6] |= 1ULL << (j & 63);
        }
    }
    mirror_lower(bits, N, stride);
    return 0;
}

/* 64-bit FNV-1a over the words, to record which bitset a stored value belongs to. */
uint64_t csg_gen_hash(const uint64_t *bits, int64_t nwords)
{
    uint64_t h = 0xCBF29CE484222325ULL;
    for (int64_t w = 0; w < nwords; ++w) {
        h ^= bits[w];
        h *= 0x100000001B3ULL;
    }
    return h;
}
