// Block occupancy of the relation matrix: which 256-row x 256-column blocks hold no relation at all.
//
// Why (Alg. 5 l.4-5: the paper's pair loop skips unrelated pairs; the run time depends
// on the ordering fraction).  The tensor kernel cannot skip single pairs, but a stage of its K sweep is the product
// of block (I, K) of the operand U and block (J, K) of the operand L, and it contributes nothing when either block
// is empty.  In a time-sorted sprinkling into a 3+1 diamond the blocks next to the diagonal are empty (elements
// that are close in time are almost never timelike separated), i.e. the first stages of every tile have an empty U
// block and the last ones an empty L block: at N = 131072 11 % of all two-stage groups are dead.  In 1+1 dimensions
// nothing is empty and the pass costs one read of the matrix (< 0.2 % of the action).
//
// occ: nB rows (nB = ceil(N / 256)) of occ_stride 32-bit words; bit (K mod 32) of word K / 32 of row I is set iff
// some bit of rows 256 I .. 256 I + 255, columns 256 K .. 256 K + 255 is set.  Every word of a row is written (words
// beyond the last column block as zero), so the buffer needs no memset.  HBM-bound: one coalesced read of the matrix
// (0.295 ms for 2 GiB).
#pragma once
#include <cstdint>

namespace csg {

constexpr int OCC_THREADS = 256;                       // 8 warps; a thread owns 16 bytes (128 columns) of every row
constexpr int OCC_WORDS_PER_CTA = OCC_THREADS / 64;    // 128 column blocks = 4 output words per CTA
constexpr int OCC_ROWS = 256;
constexpr int OCC_PAD_WORDS = 4;                       // zero words after the last column block (the kernel reads 2 ahead)

// occ_stride for N: a multiple of 4 words (one CTA writes 4), at least ceil(nB / 32) + OCC_PAD_WORDS.
__host__ __device__ inline int occ_stride_words(long long N) {
    const int nB = (int)((N + 255) / 256);
    return (((nB + 31) / 32 + OCC_PAD_WORDS + 3) / 4) * 4;
}

// grid = (occ_stride / 4, number of row blocks): CTA (c, y) reduces the rows of block I = block0 + y over column blocks
// 128 c .. 128 c + 127.  block0 > 0: the host-matrix pipeline marks the row blocks of one chunk as soon as it has landed.
__global__ void __launch_bounds__(OCC_THREADS)
occupancy_kernel(const uint64_t* __restrict__ rel, long long N, long long stride_words, uint32_t* __restrict__ occ,
                 int occ_stride, int block0) {
    __shared__ uint32_t part[OCC_THREADS / 32];
    const int I = block0 + blockIdx.y;
    const long long row0 = (long long)I * OCC_ROWS;
    const int nrows = (int)min((long long)OCC_ROWS, N - row0);
    const long long q = (long long)blockIdx.x * OCC_THREADS + threadIdx.x;     // 16-byte chunk of the row
    const bool inside = 2 * q < stride_words;
    uint4 acc = make_uint4(0u, 0u, 0u, 0u);
    if (inside) {
        const uint4* p = reinterpret_cast<const uint4*>(rel + row0 * stride_words) + q;
        const long long pitch = stride_words / 2;                               // row pitch in 16-byte units
        int r = 0;
        for (; r + 8 <= nrows; r += 8) {                                        // 8 independent loads in flight
            uint4 v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = __ldg(p + (long long)(r + u) * pitch);
#pragma unroll
            for (int u = 0; u < 8; ++u) { acc.x |= v[u].x; acc.y |= v[u].y; acc.z |= v[u].z; acc.w |= v[u].w; }
        }
        for (; r < nrows; ++r) {
            const uint4 v = __ldg(p + (long long)r * pitch);
            acc.x |= v.x; acc.y |= v.y; acc.z |= v.z; acc.w |= v.w;
        }
    }
    // two neighbouring threads hold the two halves of one 256-column block
    const uint32_t half = __ballot_sync(0xFFFFFFFFu, (acc.x | acc.y | acc.z | acc.w) != 0u);
    uint32_t b = (half | (half >> 1)) & 0x55555555u;      // bit 2m = block m of this warp; compress the even bits
    b = (b | (b >> 1)) & 0x33333333u;
    b = (b | (b >> 2)) & 0x0F0F0F0Fu;
    b = (b | (b >> 4)) & 0x00FF00FFu;
    b = (b | (b >> 8)) & 0x0000FFFFu;
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = b;                    // 16 blocks per warp
    __syncthreads();
    if (threadIdx.x < OCC_WORDS_PER_CTA) {
        const int w = OCC_WORDS_PER_CTA * blockIdx.x + threadIdx.x;
        if (w < occ_stride) occ[(long long)I * occ_stride + w] = part[2 * threadIdx.x] | (part[2 * threadIdx.x + 1] << 16);
    }
}

}  // namespace csg
