// Linking kernel: time-sorted coordinates -> packed symmetric relation matrix (the layout csg_action reads).
//
// What it computes (Sec. 2.2/2.2.2: dense adjacency matrix of the pairs that are timelike
// separated, symmetric, no self loops, elements sorted by time; the de Sitter test used by the
// paper's CUDA kernel).  The paper's GPU kernels gave one pair, later four pairs, to a thread
// of a 128-thread block, staged (d+1) floats per element in 48 KB of shared memory and shipped tiles of the
// matrix over PCIe.  Here the matrix never leaves HBM and the cost is the double-precision pair test itself:
//   * a CTA owns a 256 x 256 tile of pairs (I <= J in 256-element blocks) and stages both coordinate blocks
//     in shared memory as structure-of-arrays (conflict-free 64-bit reads);
//   * a warp owns 32 rows i; a lane owns two columns j (32 apart) of a 64-column sub-block and keeps their
//     coordinates in registers, the row's coordinates are broadcast reads; one __ballot_sync per 32 pairs
//     yields the packed word of row i, and each lane ORs its own bit into the word of the TRANSPOSED entry, so a
//     pair is tested once and lands in both triangles;
//   * the upper-triangle words leave as one 32-byte segment per row per tile, the mirrored words are transposed
//     through shared memory and leave the same way; padding columns are written as zeros.
// Arithmetic is double with one rounding per operation (__dsub_rn / __dmul_rn / __dadd_rn are never contracted
// into FMAs), in the order DESIGN.md's input recipe states, so the bits equal the host generator's bit for bit.
// 3+1 Minkowski: a single-precision test with a proven certainty bound decides the pairs far from the light cone
// (all but ~1 in 10^4) and the double-precision code decides the rest (timelike_m4_fast below): same bits.
#pragma once
#include <cstdint>

namespace csg {

constexpr int LK_T = 256;          // tile edge (elements)
constexpr int LK_THREADS = 256;
constexpr int GEOM_M2 = 0, GEOM_M4 = 1, GEOM_DS2 = 2;

template <int GEOM>
struct LinkTraits {
    static constexpr int DIM = GEOM == GEOM_M4 ? 4 : 2;
};

// Is the earlier element a (coordinates a[]) related to the later element b?  Branch-free.
template <int GEOM>
__device__ __forceinline__ bool timelike(const double* a, const double* b) {
    if (GEOM == GEOM_M2) {
        return (a[0] < b[0]) & (a[1] < b[1]);
    } else if (GEOM == GEOM_M4) {
        const double dt = __dsub_rn(b[0], a[0]), dx = __dsub_rn(b[1], a[1]);
        const double dy = __dsub_rn(b[2], a[2]), dz = __dsub_rn(b[3], a[3]);
        double s2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
        s2 = __dadd_rn(s2, __dmul_rn(dz, dz));
        // dt > 0.0 on the integer pipe: a double is > 0 iff its bit pattern, read as a signed integer, is > 0
        // (a positive NaN passes here and fails the next comparison, as it does in "dt > 0.0 && ...")
        return (__double_as_longlong(dt) > 0LL) & (__dmul_rn(dt, dt) > s2);
    } else {
        const double PI = 3.14159265358979323846;
        const double dth = fabs(__dsub_rn(a[1], b[1]));
        const double lhs = __dsub_rn(PI, fabs(__dsub_rn(PI, dth)));
        return lhs < fabs(__dsub_rn(a[0], b[0]));
    }
}

// GEOM_M4 fast path.  Double precision is the scarce pipe (64 lanes per clock per SM against 128 for single), and
// almost every pair is far from the light cone, where single precision already decides.  With every coordinate of the
// tile bounded by M, the single-precision value s_f of dt^2 - (dx^2 + dy^2 + dz^2) differs from the exact one by at
// most 2^-17 M^2: the four differences carry 2^-22 M each (conversion of both coordinates 2 x 2^-24 M, the
// subtraction 2^-24 x 2M), their squares therefore 4 x 2^-20 M^2 in all, and the four roundings of the sum of
// magnitudes <= 16 M^2 another 2^-18 M^2; the double-precision test itself is off by ~10^-15 M^2.  So |s_f| > E :=
// 2^-16 M^2 fixes the sign of the exact expression and of the double test (and s_f > E implies |dt| > 2^-8.5 M, far
// above the 2^-22 M uncertainty of dt_f, so the sign of dt_f is the sign of dt); everything else -- about one pair in 10^4, NaNs
// included -- is decided by the double-precision code above, for the whole warp step.  Bit-identical by construction;
// checked word for word against the plain CPU linking code of the tests and the host generator (tests/test_gpu_link.py).  M outside [1e-10, 1e15]
// (single-precision underflow or overflow of the squares) switches the fast path off for the tile (E = +inf).
__device__ __forceinline__ void timelike_m4_fast(const float4& r, const float4& a, float E, bool& related, bool& unsure) {
    const float dt = __fsub_rn(a.x, r.x), dx = __fsub_rn(a.y, r.y), dy = __fsub_rn(a.z, r.z), dz = __fsub_rn(a.w, r.w);
    float q = __fmul_rn(dx, dx);
    q = __fmaf_rn(dy, dy, q);
    q = __fmaf_rn(dz, dz, q);
    // dt |dt| instead of dt^2 (|dt| is an operand modifier, not an instruction): a pair with dt < 0 -- only possible when
    // the input is not time-sorted -- lands below -E or in the uncertain band, never above E, so "dt > 0" needs no test
    const float sf = __fmaf_rn(dt, fabsf(dt), -q);
    related = sf > E;
    unsure = !(fabsf(sf) > E);
}

// low `n` bits set (n clamped to 0..32)
__device__ __forceinline__ uint32_t low_bits(long long n) {
    return n <= 0 ? 0u : (n >= 32 ? 0xFFFFFFFFu : ((1u << (int)n) - 1u));
}

// coords: N x DIM doubles, one row per element, sorted by time.  rel: N rows of stride64 words, every word
// of every row is written (zero padding).  Grid: one CTA per tile t = (I, J), I <= J, row-major over I.
// The pair loop tests every (row, column) of the tile as (earlier, later) with no bounds or order checks; rows
// and columns beyond N, and the lower triangle of a diagonal tile (where "earlier" is wrong), are masked
// off the packed words afterwards.
template <int GEOM>
__global__ void __launch_bounds__(LK_THREADS, 2)
link_kernel(const double* __restrict__ coords, long long N, long long stride64, uint64_t* __restrict__ rel, int nB) {
    constexpr int DIM = LinkTraits<GEOM>::DIM;
    __shared__ double ci[DIM][LK_T];
    __shared__ double cj[DIM][LK_T];
    __shared__ uint32_t tr[LK_T][8 + 1];   // transposed words: row j, 32-bit word w (+1: bank spread)
    __shared__ float4 fi[GEOM == GEOM_M4 ? LK_T : 1];   // rows in single precision (GEOM_M4 fast path)
    __shared__ float mred[LK_THREADS / 32];

    // tile index -> (I, J): row I of the upper triangle holds nB - I tiles, I nB - I(I-1)/2 tiles come
    // before it; closed form, then corrected for the rounding of the square root
    const long long t = blockIdx.x, b2 = 2LL * nB + 1;
    int I = (int)(((double)b2 - sqrt((double)(b2 * b2 - 8 * t))) * 0.5);
    I = max(0, min(I, nB - 1));
    while (I > 0 && (long long)I * nB - (long long)I * (I - 1) / 2 > t) --I;
    while ((long long)(I + 1) * nB - (long long)(I + 1) * I / 2 <= t) ++I;
    const int J = I + (int)(t - ((long long)I * nB - (long long)I * (I - 1) / 2));
    const long long i0 = (long long)I * LK_T, j0 = (long long)J * LK_T;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const bool diag = I == J;

    float E = 0.0f;                          // GEOM_M4: certainty bound of the single-precision test
    {   // stage coordinates (rows beyond N: zeros, masked below)
        const long long ri = i0 + tid, rj = j0 + tid;
        float m = 0.0f;
#pragma unroll
        for (int c = 0; c < DIM; ++c) {
            const double vi = ri < N ? coords[ri * DIM + c] : 0.0, vj = rj < N ? coords[rj * DIM + c] : 0.0;
            ci[c][tid] = vi;
            cj[c][tid] = vj;
            if (GEOM == GEOM_M4) m = fmaxf(m, fmaxf(__double2float_ru(fabs(vi)), __double2float_ru(fabs(vj))));   // NaN: ignored here, caught per pair
        }
        if (GEOM == GEOM_M4) {
            fi[tid] = make_float4((float)ci[0][tid], (float)ci[1][tid], (float)ci[2][tid], (float)ci[3][tid]);
            m = __uint_as_float(__reduce_max_sync(0xFFFFFFFFu, __float_as_uint(m)));   // non-negative floats order like their bit patterns
            if ((tid & 31) == 0) mred[tid >> 5] = m;
        }
    }
    __syncthreads();
    if (GEOM == GEOM_M4) {
        float M = 0.0f;
#pragma unroll
        for (int w = 0; w < LK_THREADS / 32; ++w) M = fmaxf(M, mred[w]);
        E = (M >= 1e-10f && M <= 1e15f) ? __fmul_ru(__fmul_ru(M, M), 1.52587890625e-05f) : __int_as_float(0x7f800000);
    }

    const int row_l = 32 * warp + lane;                       // this thread's row of the tile (= tid)
    const uint32_t rows_ok = low_bits(N - (i0 + 32 * warp));  // rows 32 warp + ii of this warp that exist
    uint32_t direct[8];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
        const int ja = 64 * s + lane, jb = ja + 32;           // columns inside the tile
        double a[DIM], b[DIM];
#pragma unroll
        for (int c = 0; c < DIM; ++c) { a[c] = cj[c][ja]; b[c] = cj[c][jb]; }
        float4 af = make_float4(0.f, 0.f, 0.f, 0.f), bf = af;
        if (GEOM == GEOM_M4) {
            af = make_float4((float)a[0], (float)a[1], (float)a[2], (float)a[3]);
            bf = make_float4((float)b[0], (float)b[1], (float)b[2], (float)b[3]);
        }
        uint32_t ta = 0u, tb = 0u, keep_lo = 0u, keep_hi = 0u;
#pragma unroll 1
        for (int i8 = 0; i8 < 32; i8 += 8) {
            uint32_t pa8 = 0u, pb8 = 0u;
            if (GEOM == GEOM_M4) {
                // eight rows in single precision, straight-line (16 independent pair tests per thread); the rows in which
                // some lane's pair was too close to the cone are redone in double precision afterwards (rare)
                uint32_t un8 = 0u;
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    bool pa, pb, ua, ub;
                    const float4 rf = fi[32 * warp + i8 + k];
                    timelike_m4_fast(rf, af, E, pa, ua);
                    timelike_m4_fast(rf, bf, E, pb, ub);
                    const uint32_t wa = __ballot_sync(0xFFFFFFFFu, pa), wb = __ballot_sync(0xFFFFFFFFu, pb);
                    if (lane == i8 + k) { keep_lo = wa; keep_hi = wb; }
                    pa8 |= pa ? (1u << k) : 0u;
                    pb8 |= pb ? (1u << k) : 0u;
                    un8 |= (ua | ub) ? (1u << k) : 0u;
                }
                uint32_t fix = __reduce_or_sync(0xFFFFFFFFu, un8);
                while (fix) {
                    const int k = __ffs((int)fix) - 1;
                    fix &= fix - 1;
                    const int il = 32 * warp + i8 + k;
                    double r[DIM];
#pragma unroll
                    for (int c = 0; c < DIM; ++c) r[c] = ci[c][il];
                    const bool pa = timelike<GEOM>(r, a), pb = timelike<GEOM>(r, b);
                    const uint32_t wa = __ballot_sync(0xFFFFFFFFu, pa), wb = __ballot_sync(0xFFFFFFFFu, pb);
                    if (lane == i8 + k) { keep_lo = wa; keep_hi = wb; }
                    pa8 = (pa8 & ~(1u << k)) | (pa ? (1u << k) : 0u);
                    pb8 = (pb8 & ~(1u << k)) | (pb ? (1u << k) : 0u);
                }
            } else {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int il = 32 * warp + i8 + k;            // row inside the tile
                    double r[DIM];
#pragma unroll
                    for (int c = 0; c < DIM; ++c) r[c] = ci[c][il];
                    const bool pa = timelike<GEOM>(r, a), pb = timelike<GEOM>(r, b);
                    const uint32_t wa = __ballot_sync(0xFFFFFFFFu, pa), wb = __ballot_sync(0xFFFFFFFFu, pb);
                    if (lane == i8 + k) { keep_lo = wa; keep_hi = wb; }
                    pa8 |= pa ? (1u << k) : 0u;
                    pb8 |= pb ? (1u << k) : 0u;
                }
            }
            ta |= pa8 << i8;
            tb |= pb8 << i8;
        }
        // masks: existing columns / rows; on a diagonal tile keep column > row only
        uint32_t ca = low_bits(N - (j0 + 64 * s)), cb = low_bits(N - (j0 + 64 * s + 32));
        uint32_t ra = rows_ok, rb = rows_ok;
        if (diag) {
            ca &= ~low_bits(row_l + 1 - 64 * s);               // columns 64 s + bit > row_l
            cb &= ~low_bits(row_l + 1 - 64 * s - 32);
            ra &= low_bits(ja - 32 * warp);                    // rows 32 warp + bit < ja
            rb &= low_bits(jb - 32 * warp);
        }
        direct[2 * s] = keep_lo & ca;
        direct[2 * s + 1] = keep_hi & cb;
        tr[ja][warp] = ta & ra;
        tr[jb][warp] = tb & rb;
    }
    __syncthreads();
    if (diag) {   // both triangles land in the same 256 x 256 block: row tid = upper words | mirrored words
#pragma unroll
        for (int w = 0; w < 8; ++w) direct[w] |= tr[tid][w];
    }
    const long long row = i0 + tid;
    if (row < N) {   // upper-triangle words: row i0 + tid, words 4J..4J+3
        uint4* dst = reinterpret_cast<uint4*>(rel + row * stride64 + 4 * J);
        dst[0] = make_uint4(direct[0], direct[1], direct[2], direct[3]);
        dst[1] = make_uint4(direct[4], direct[5], direct[6], direct[7]);
    }
    const long long rowj = j0 + tid;
    if (!diag && rowj < N) {   // mirrored words: row j0 + tid, words 4I..4I+3
        uint4* dst = reinterpret_cast<uint4*>(rel + rowj * stride64 + 4 * I);
        dst[0] = make_uint4(tr[tid][0], tr[tid][1], tr[tid][2], tr[tid][3]);
        dst[1] = make_uint4(tr[tid][4], tr[tid][5], tr[tid][6], tr[tid][7]);
    }
}

}  // namespace csg
