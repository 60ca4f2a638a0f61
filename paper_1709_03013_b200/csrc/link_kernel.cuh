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

    {   // stage coordinates (rows beyond N: zeros, masked below)
        const long long ri = i0 + tid, rj = j0 + tid;
#pragma unroll
        for (int c = 0; c < DIM; ++c) {
            ci[c][tid] = ri < N ? coords[ri * DIM + c] : 0.0;
            cj[c][tid] = rj < N ? coords[rj * DIM + c] : 0.0;
        }
    }
    __syncthreads();

    const int row_l = 32 * warp + lane;                       // this thread's row of the tile (= tid)
    const uint32_t rows_ok = low_bits(N - (i0 + 32 * warp));  // rows 32 warp + ii of this warp that exist
    uint32_t direct[8];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
        const int ja = 64 * s + lane, jb = ja + 32;           // columns inside the tile
        double a[DIM], b[DIM];
#pragma unroll
        for (int c = 0; c < DIM; ++c) { a[c] = cj[c][ja]; b[c] = cj[c][jb]; }
        uint32_t ta = 0u, tb = 0u, keep_lo = 0u, keep_hi = 0u;
#pragma unroll 1
        for (int i8 = 0; i8 < 32; i8 += 8) {
            uint32_t pa8 = 0u, pb8 = 0u;
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
