// Bitset variant of the interval kernel: AND + POPC over packed 32-bit words.
//
// What it computes (Sec. 4.1, Fig. 2, Alg. 5 l.7): for every related
// pair i<j, n_ij = popcount(R[i] & R[j]) over bit columns i+1..j-1, bucketed into counts[n_ij].
// The paper walks pairs one at a time on a CPU core (Alg. 5) and re-reads both rows for every pair; here a
// CTA owns a 64x64 tile of pairs, stages the 64+64 row segments of a 1024-column K-chunk in shared memory
// once, and every thread keeps a 4x4 register micro-tile of partial popcounts, so each staged word is used
// 64 times.  The open range i<k<j is applied when a row segment is staged: row i keeps only columns > i
// (operand "U"), row j keeps only columns < j (operand "L"), so n_ij = sum_k U[i][k] & L[j][k] with no
// per-pair masking in the inner loop.
//
// Small sets are launch-bound (N = 1024: ~14 us of kernel), so for them the memset before and the finishing kernel
// after are folded into this launch (`fused` != NULL): CTAs add their histograms into a zeroed library workspace, the
// last CTA to finish (a ticket) moves the sums to `counts`, re-zeroes the workspace for the next launch on the same
// stream and computes S (finish.cuh).
#pragma once
#include <cstdint>

#include "finish.cuh"

namespace csg {

constexpr int BS_T = 64;         // tile edge in pairs
constexpr int BS_KW = 32;        // 32-bit words per K-chunk
constexpr int BS_LD = 36;        // shared row stride in words (32 + 4 pad: conflict-free 128-bit reads)
constexpr int BS_THREADS = 256;
constexpr int BS_HIST = 2048;    // privatised low bins per CTA
constexpr int BS_FUSED_BINS = 1024;   // fused single-launch path: kmax + 1 <= this (N <= 1024 under CSG_VARIANT_AUTO)

// Workspace of the fused path, one per stream (launches on one stream run one after the other): all zero between launches.
struct BitsetFusedWs {
    unsigned long long acc[BS_FUSED_BINS];
    unsigned int ticket;
};

// Bits of 32-bit word kw (columns 32kw..32kw+31) with column index > i.
__device__ __forceinline__ uint32_t mask_cols_gt(long long i, long long kw) {
    long long lo = kw * 32;
    if (lo > i) return 0xFFFFFFFFu;
    if (lo + 31 <= i) return 0u;
    return 0xFFFFFFFFu << (int)(i - lo + 1);
}
// Bits of 32-bit word kw with column index < j.
__device__ __forceinline__ uint32_t mask_cols_lt(long long j, long long kw) {
    long long lo = kw * 32;
    if (lo + 31 < j) return 0xFFFFFFFFu;
    if (lo >= j) return 0u;
    return (1u << (int)(j - lo)) - 1u;
}

// Tiles (I,J), I<=J, in 64-row units, enumerated by descending K-depth d=J-I (longest first).
__device__ __forceinline__ void bitset_tile_from_index(long long t, long long nb, long long& I, long long& J) {
    long long m = (long long)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((m + 1) * (m + 2) / 2 <= t) ++m;
    while (m * (m + 1) / 2 > t) --m;
    long long d = nb - 1 - m;
    I = t - m * (m + 1) / 2;
    J = I + d;
}

__global__ void __launch_bounds__(BS_THREADS, 2)
bitset_action_kernel(const uint32_t* __restrict__ rel, long long N, long long stride32, int kmax,
                     unsigned long long* __restrict__ counts, long long nb, long long ntiles, int shard,
                     int nshards, long long set_stride32, long long counts_stride, BitsetFusedWs* __restrict__ fused,
                     int dim, double eps, double* __restrict__ S) {
    // blockIdx.y = causal set of a batch (csg_action_batch): same N, matrices set_stride32 words apart
    rel += (long long)blockIdx.y * set_stride32;
    counts += (long long)blockIdx.y * counts_stride;
    __shared__ __align__(16) uint32_t sA[BS_T * BS_LD];
    __shared__ __align__(16) uint32_t sB[BS_T * BS_LD];
    __shared__ unsigned int hist[BS_HIST];

    const int tid = threadIdx.x;
    const int ty = tid >> 4, tx = tid & 15;
    for (int b = tid; b < BS_HIST; b += BS_THREADS) hist[b] = 0u;
    __syncthreads();

    // this launch owns the tiles t = shard (mod nshards) of the depth-sorted enumeration
    for (long long t = shard + (long long)blockIdx.x * nshards; t < ntiles; t += (long long)gridDim.x * nshards) {
        long long I, J;
        bitset_tile_from_index(t, nb, I, J);
        const long long i0 = I * BS_T, j0 = J * BS_T;
        const long long kw_begin = (i0 >> 5) & ~3LL;               // 16-byte aligned start
        const long long kw_end = ((j0 + BS_T - 1) >> 5) + 1;       // exclusive

        int acc[4][4];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) acc[a][b] = 0;

        for (long long kw0 = kw_begin; kw0 < kw_end; kw0 += BS_KW) {
            // stage 64 rows x 32 words of each operand, masked to the open range
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int r = (tid >> 3) + 32 * h;
                const long long kw = kw0 + 4 * (tid & 7);
                const bool in_row = (kw + 3 < stride32) && (kw < kw_end);
                uint4 va = make_uint4(0, 0, 0, 0), vb = make_uint4(0, 0, 0, 0);
                const long long ri = i0 + r, rj = j0 + r;
                if (in_row && ri < N) {
                    va = __ldg(reinterpret_cast<const uint4*>(rel + ri * stride32 + kw));
                    va.x &= mask_cols_gt(ri, kw);
                    va.y &= mask_cols_gt(ri, kw + 1);
                    va.z &= mask_cols_gt(ri, kw + 2);
                    va.w &= mask_cols_gt(ri, kw + 3);
                }
                if (in_row && rj < N) {
                    vb = __ldg(reinterpret_cast<const uint4*>(rel + rj * stride32 + kw));
                    vb.x &= mask_cols_lt(rj, kw);
                    vb.y &= mask_cols_lt(rj, kw + 1);
                    vb.z &= mask_cols_lt(rj, kw + 2);
                    vb.w &= mask_cols_lt(rj, kw + 3);
                }
                *reinterpret_cast<uint4*>(&sA[r * BS_LD + 4 * (tid & 7)]) = va;
                *reinterpret_cast<uint4*>(&sB[r * BS_LD + 4 * (tid & 7)]) = vb;
            }
            __syncthreads();
            // only the 128-bit quads that hold columns of this tile's K range (short ranges dominate at small N)
            const int nq = (int)min((long long)(BS_KW / 4), (kw_end - kw0 + 3) >> 2);
#pragma unroll 2
            for (int kq = 0; kq < nq; ++kq) {
                uint4 a4[4], b4[4];
#pragma unroll
                for (int a = 0; a < 4; ++a)
                    a4[a] = *reinterpret_cast<const uint4*>(&sA[(4 * ty + a) * BS_LD + 4 * kq]);
#pragma unroll
                for (int b = 0; b < 4; ++b)
                    b4[b] = *reinterpret_cast<const uint4*>(&sB[(tx + 16 * b) * BS_LD + 4 * kq]);
#pragma unroll
                for (int a = 0; a < 4; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b)
                        acc[a][b] += __popc(a4[a].x & b4[b].x) + __popc(a4[a].y & b4[b].y) +
                                     __popc(a4[a].z & b4[b].z) + __popc(a4[a].w & b4[b].w);
            }
            __syncthreads();
        }

        // fused epilogue: mask by R[i][j] (and i<j), bucket n_ij
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            const long long i = i0 + 4 * ty + a;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const long long j = j0 + tx + 16 * b;
                if (i < j && j < N) {
                    const uint32_t w = __ldg(rel + i * stride32 + (j >> 5));
                    const int n = acc[a][b];
                    if (((w >> (j & 31)) & 1u) && n <= kmax) {
                        if (n < BS_HIST) atomicAdd(&hist[n], 1u);
                        else atomicAdd(&counts[n], 1ULL);
                    }
                }
            }
        }
    }

    __syncthreads();
    unsigned long long* const target = fused ? fused->acc : counts;
    for (int b = tid; b < BS_HIST && b <= kmax; b += BS_THREADS)
        if (hist[b]) atomicAdd(&target[b], (unsigned long long)hist[b]);
    if (fused == nullptr) return;
    // ---- fused tail (single set, kmax < BS_FUSED_BINS): the last CTA publishes counts and S
    __shared__ unsigned int is_last;
    __threadfence();                                  // this CTA's sums are visible before its ticket is
    __syncthreads();
    if (tid == 0) is_last = atomicAdd(&fused->ticket, 1u) == gridDim.x - 1 ? 1u : 0u;
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    long long* sums = reinterpret_cast<long long*>(sB);          // 9216 bytes >= BS_FUSED_BINS x 8
    double* red = reinterpret_cast<double*>(sA);                 // 9216 bytes >= FIN_LANES x 8
    for (int b = tid; b < BS_FUSED_BINS; b += BS_THREADS) {
        const unsigned long long v = b <= kmax ? atomicExch(&fused->acc[b], 0ULL) : 0ULL;   // read and re-zero
        sums[b] = (long long)v;
        if (b <= kmax) counts[b] = v;
    }
    if (tid == 0) fused->ticket = 0u;
    __syncthreads();
    finish_block(sums, N, dim, eps, kmax, S, red);
}

// Test hook (csg_interval_sizes): one warp per listed pair, straight AND+POPC over the open range.
__global__ void pair_interval_kernel(const uint32_t* __restrict__ rel, long long N, long long stride32,
                                     const long long* __restrict__ pairs, long long npairs,
                                     int* __restrict__ n_out) {
    const long long p = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (p >= npairs) return;
    const long long i = pairs[2 * p], j = pairs[2 * p + 1];
    int result = -1;
    if (i >= 0 && i < j && j < N) {
        const uint32_t wij = __ldg(rel + i * stride32 + (j >> 5));
        if ((wij >> (j & 31)) & 1u) {
            int n = 0;
            for (long long kw = (i >> 5) + lane; kw <= (j >> 5); kw += 32) {
                uint32_t w = __ldg(rel + i * stride32 + kw) & __ldg(rel + j * stride32 + kw);
                w &= mask_cols_gt(i, kw) & mask_cols_lt(j, kw);
                n += __popc(w);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xFFFFFFFFu, n, o);
            result = n;
        }
    }
    if (lane == 0) n_out[p] = result;
}

}  // namespace csg
