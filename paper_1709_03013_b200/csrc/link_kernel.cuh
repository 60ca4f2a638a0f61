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
// into FMAs), in the order DESIGN.md's input recipe states, so the bits equal the host generator's and the
// oracle's bit for bit.
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

// Is the earlier element a (coordinates a[]) related to the later element b?
template <int GEOM>
__device__ __forceinline__ bool timelike(const double* a, const double* b) {
    if (GEOM == GEOM_M2) {
        return a[0] < b[0] && a[1] < b[1];
    } else if (GEOM == GEOM_M4) {
        const double dt = __dsub_rn(b[0], a[0]), dx = __dsub_rn(b[1], a[1]);
        const double dy = __dsub_rn(b[2], a[2]), dz = __dsub_rn(b[3], a[3]);
        double s2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
        s2 = __dadd_rn(s2, __dmul_rn(dz, dz));
        return dt > 0.0 && __dmul_rn(dt, dt) > s2;
    } else {
        const double PI = 3.14159265358979323846;
        const double dth = fabs(__dsub_rn(a[1], b[1]));
        const double lhs = __dsub_rn(PI, fabs(__dsub_rn(PI, dth)));
        return lhs < fabs(__dsub_rn(a[0], b[0]));
    }
}

// coords: N x DIM doubles, one row per element, sorted by time.  rel: N rows of stride64 words, every word
// of every row is written (zero padding).  Grid: one CTA per tile t = (I, J), I <= J, row-major over I.
template <int GEOM>
__global__ void __launch_bounds__(LK_THREADS, 2)
link_kernel(const double* __restrict__ coords, long long N, long long stride64, uint64_t* __restrict__ rel, int nB) {
    constexpr int DIM = LinkTraits<GEOM>::DIM;
    __shared__ double ci[DIM][LK_T];
    __shared__ double cj[DIM][LK_T];
    __shared__ __align__(16) uint32_t tr[LK_T][8 + 1];   // transposed words: row j, 32-bit word w (+1: bank spread)

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

    uint64_t direct[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
        const int ja = 64 * s + lane, jb = ja + 32;           // columns inside the tile
        double a[DIM], b[DIM];
#pragma unroll
        for (int c = 0; c < DIM; ++c) { a[c] = cj[c][ja]; b[c] = cj[c][jb]; }
        const bool va = j0 + ja < N, vb = j0 + jb < N;
        uint32_t ta = 0u, tb = 0u, keep_lo = 0u, keep_hi = 0u;
#pragma unroll 8
        for (int ii = 0; ii < 32; ++ii) {
            const int il = 32 * warp + ii;                    // row inside the tile
            double r[DIM];
#pragma unroll
            for (int c = 0; c < DIM; ++c) r[c] = ci[c][il];
            const bool vi = i0 + il < N;
            bool pa, pb;
            if (!diag) {
                pa = vi && va && timelike<GEOM>(r, a);
                pb = vi && vb && timelike<GEOM>(r, b);
            } else {                                           // both triangles of a diagonal tile, earlier element first
                pa = vi && va && (il < ja ? timelike<GEOM>(r, a) : (il > ja && timelike<GEOM>(a, r)));
                pb = vi && vb && (il < jb ? timelike<GEOM>(r, b) : (il > jb && timelike<GEOM>(b, r)));
            }
            const uint32_t wa = __ballot_sync(0xFFFFFFFFu, pa), wb = __ballot_sync(0xFFFFFFFFu, pb);
            if (lane == ii) { keep_lo = wa; keep_hi = wb; }
            ta |= (pa ? 1u : 0u) << ii;
            tb |= (pb ? 1u : 0u) << ii;
        }
        direct[s] = (uint64_t)keep_lo | ((uint64_t)keep_hi << 32);
        tr[ja][warp] = ta;
        tr[jb][warp] = tb;
    }
    {   // upper-triangle words: row i0 + 32 warp + lane, words 4J..4J+3
        const long long row = i0 + 32 * warp + lane;
        if (row < N) {
            uint4* dst = reinterpret_cast<uint4*>(rel + row * stride64 + 4 * J);
            dst[0] = make_uint4((uint32_t)direct[0], (uint32_t)(direct[0] >> 32), (uint32_t)direct[1], (uint32_t)(direct[1] >> 32));
            dst[1] = make_uint4((uint32_t)direct[2], (uint32_t)(direct[2] >> 32), (uint32_t)direct[3], (uint32_t)(direct[3] >> 32));
        }
    }
    if (diag) return;
    __syncthreads();
    {   // mirrored words: row j0 + tid, words 4I..4I+3
        const long long row = j0 + tid;
        if (row < N) {
            uint4* dst = reinterpret_cast<uint4*>(rel + row * stride64 + 4 * I);
            dst[0] = make_uint4(tr[tid][0], tr[tid][1], tr[tid][2], tr[tid][3]);
            dst[1] = make_uint4(tr[tid][4], tr[tid][5], tr[tid][6], tr[tid][7]);
        }
    }
}

}  // namespace csg
