// Tensor-core variant of the interval kernel: a tiled binary "GEMM" on tcgen05 (sm_100a).
//
// What it computes (Sec. 4.1, Fig. 2, Alg. 5 l.7): for every related
// pair i<j, n_ij = sum_{i<k<j} R[i][k] * R[j][k], bucketed into counts[n_ij].  With U[i][k] = R[i][k]*[k>i]
// and L[j][k] = R[j][k]*[k<j] this is the matrix product C = U * L^T restricted to the upper triangle and
// masked by R[i][j] -- a dense contraction over k, so it runs on the 5th-generation tensor cores:
//
//   * a CTA owns a 128 x 256 tile of pairs (rows i of block I, rows j of block J) and sweeps K from the
//     first column of block I to the last column of block J in stages of 128 columns;
//   * 12 producer warps read the packed bits of their row (16 bytes per row per stage, straight from
//     global/L2 with a two-stage register prefetch), expand them to 0/1 unsigned bytes and store them into a
//     4-stage ring of K-major, 128-byte-swizzled operand tiles in shared memory.  The order of the 32 k's
//     inside a 32-bit word is permuted ((w >> q) & 0x01010101 puts bits q, q+8, q+16, q+24 into one 32-bit
//     store); both operands use the same permutation and the MMA sums over k, so the result is unchanged;
//   * one thread issues tcgen05.mma.cta_group::1.kind::i8 (M=128, N=256, K=32, u8 x u8 -> s32, exact) four
//     times per stage, accumulating in 256 TMEM columns; tcgen05.commit hands the stage back to the producers;
//   * the open range i<k<j costs nothing in the steady state: only the first stage of a tile (columns of
//     block I) needs the k>i mask and only the last two stages (columns of block J) need the k<j mask;
//   * fused epilogue: the same 12 warps read the accumulators back with tcgen05.ld, test bit R[i][j] (and
//     i<j), and bucket n_ij into a privatised shared-memory histogram (low bins) or straight into the global
//     counts (high bins, smeared action only).  No N x N count matrix ever reaches HBM.
//
// Tiles are handed out statically from a list sorted by K-depth, longest first, in boustrophedon order over
// the persistent CTAs (one per SM), which balances the triangular workload without a global counter.
#pragma once
#include <cstdint>

namespace csg {

constexpr int TC_TM = 128;                 // rows i per tile (UMMA M)
constexpr int TC_TN = 256;                 // rows j per tile (UMMA N)
constexpr int TC_KS = 128;                 // k columns per stage = bytes per operand row in smem
constexpr int TC_STAGES = 4;
constexpr int TC_A_BYTES = TC_TM * TC_KS;  // 16 KiB
constexpr int TC_B_BYTES = TC_TN * TC_KS;  // 32 KiB
constexpr int TC_STAGE_BYTES = TC_A_BYTES + TC_B_BYTES;
constexpr int TC_PRODUCER_WARPS = 12;      // 4 for the A rows, 8 for the B rows
constexpr int TC_PRODUCERS = TC_PRODUCER_WARPS * 32;
constexpr int TC_THREADS = TC_PRODUCERS + 32;  // + the MMA warp
constexpr int TC_HIST = 4096;              // privatised low bins per CTA
constexpr int TC_TMEM_COLS = 256;
constexpr int TC_SMEM_BYTES = TC_STAGES * TC_STAGE_BYTES + TC_HIST * 4 + 256 + 1024;  // + barriers + align

// ---------------------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// D[tmem] (+)= A[smem] * B[smem]^T, u8 x u8 -> s32, one CTA.
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                        uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d), "l"(adesc), "l"(bdesc),
        "r"(idesc), "r"(accumulate) : "memory");
}
// Arrive on an mbarrier once all tcgen05 ops issued so far by this thread have completed.
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar)
                 : "memory");
}
// 32 lanes x 32 consecutive 32-bit columns: thread t of the warp gets lane (base+t), columns c..c+31.
__device__ __forceinline__ void tmem_ld_32x32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]),
          "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]),
          "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]),
          "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Shared-memory matrix descriptor: K-major operand, 128-byte swizzle, rows of 128 bytes, 8-row groups
// 1024 bytes apart (SBO), descriptor version 1 (sm_100).
__device__ __forceinline__ uint64_t make_kmajor_sw128_desc(uint32_t smem_addr) {
    const uint32_t lo = ((smem_addr >> 4) & 0x3FFFu) | (1u << 16);           // start address, LBO = 1 (unused)
    const uint32_t hi = (1024u >> 4) | (1u << 14) | (2u << 29);              // SBO, version, SWIZZLE_128B
    return (static_cast<uint64_t>(hi) << 32) | lo;
}
// Instruction descriptor, kind::i8: D = s32, A = B = u8, both K-major, N = 256, M = 128.
constexpr uint32_t TC_IDESC = (2u << 4) | ((TC_TN >> 3) << 17) | ((TC_TM >> 4) << 24);

// One row's 128 k-bits (4 words) -> 128 bytes in the swizzled operand row.
__device__ __forceinline__ void unpack_row_to_smem(uint8_t* tile, int r, const uint4& w) {
    uint8_t* row = tile + (r >> 3) * 1024 + (r & 7) * 128;
    const int sw = r & 7;
    const uint32_t ws[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const uint32_t x = ws[m];
        uint4 lo, hi;
        lo.x = x & 0x01010101u;
        lo.y = (x >> 1) & 0x01010101u;
        lo.z = (x >> 2) & 0x01010101u;
        lo.w = (x >> 3) & 0x01010101u;
        hi.x = (x >> 4) & 0x01010101u;
        hi.y = (x >> 5) & 0x01010101u;
        hi.z = (x >> 6) & 0x01010101u;
        hi.w = (x >> 7) & 0x01010101u;
        *reinterpret_cast<uint4*>(row + (((2 * m) ^ sw) << 4)) = lo;
        *reinterpret_cast<uint4*>(row + (((2 * m + 1) ^ sw) << 4)) = hi;
    }
}

// keep local bit positions p (0..127) with p > r   (operand U in the stage that holds row i's own column)
__device__ __forceinline__ uint32_t keep_gt(int r, int m) {
    const int s = r - 32 * m + 1;  // number of low bits to clear
    return s <= 0 ? 0xFFFFFFFFu : (s >= 32 ? 0u : (0xFFFFFFFFu << s));
}
// keep local bit positions p with p < lim   (operand L in the stages that hold row j's own column)
__device__ __forceinline__ uint32_t keep_lt(int lim, int m) {
    const int s = lim - 32 * m;    // number of low bits to keep
    return s <= 0 ? 0u : (s >= 32 ? 0xFFFFFFFFu : ((1u << s) - 1u));
}

// tile list entry: I (128-row block) in the low 16 bits... kept as int2 {I, J} for clarity.
__global__ void __launch_bounds__(TC_THREADS, 1)
tensor_action_kernel(const uint64_t* __restrict__ rel, long long N, long long stride_words, int kmax,
                     unsigned long long* __restrict__ counts, const int2* __restrict__ tiles, int ntiles) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* stage_base = smem;
    unsigned int* hist = reinterpret_cast<unsigned int*>(smem + TC_STAGES * TC_STAGE_BYTES);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + TC_STAGES * TC_STAGE_BYTES + TC_HIST * 4);
    // bars[0..3] full, bars[4..7] empty, bars[8] tmem_full, bars[9] tmem_empty, then the TMEM base address
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 10);

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + TC_STAGES);
    const uint32_t tmem_full = smem_u32(bars + 2 * TC_STAGES), tmem_empty = smem_u32(bars + 2 * TC_STAGES + 1);

    for (int b = tid; b < TC_HIST; b += TC_THREADS) hist[b] = 0u;
    if (tid == 0) {
        for (int s = 0; s < TC_STAGES; ++s) {
            mbar_init(full0 + 8 * s, TC_PRODUCERS);
            mbar_init(empty0 + 8 * s, 1);
        }
        mbar_init(tmem_full, 1);
        mbar_init(tmem_empty, TC_PRODUCERS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == TC_PRODUCER_WARPS) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                     "n"(TC_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int G = gridDim.x, cta = blockIdx.x;
    const int rounds = (ntiles + G - 1) / G;

    if (warp < TC_PRODUCER_WARPS) {
        // ================================================================== producers + epilogue
        const bool isA = warp < 4;
        const int r = isA ? tid : tid - 128;          // row inside the A (0..127) or B (0..255) tile
        const int q4 = warp & 3;                      // TMEM lane quarter this warp may read
        const int cgrp = warp >> 2;                   // which third of the 8 column chunks it drains
        const int c_begin = cgrp * 3, c_end = cgrp == 2 ? 8 : c_begin + 3;
        uint32_t stage = 0, sphase = 0;               // ring position / parity
        uint32_t tphase = 0;                          // parity of tmem_full

        for (int rd = 0; rd < rounds; ++rd) {
            const int t = rd * G + ((rd & 1) ? (G - 1 - cta) : cta);
            if (t >= ntiles) continue;
            const int2 tile = tiles[t];
            const int I = tile.x, J = tile.y;
            const long long i0 = (long long)I * TC_TM, j0 = (long long)J * TC_TN;
            const int kb_begin = I, kb_end = 2 * J + 2;   // stages of 128 columns, [begin, end)
            const long long row = isA ? i0 + r : j0 + r;
            const bool row_ok = row < N;
            const uint4* src = reinterpret_cast<const uint4*>(rel + (row_ok ? row : 0) * stride_words);
            const uint4 zero = make_uint4(0, 0, 0, 0);

            uint4 w0 = row_ok ? __ldg(src + kb_begin) : zero;
            uint4 w1 = (row_ok && kb_begin + 1 < kb_end) ? __ldg(src + kb_begin + 1) : zero;
            for (int kb = kb_begin; kb < kb_end; ++kb) {
                uint4 w2 = (row_ok && kb + 2 < kb_end) ? __ldg(src + kb + 2) : zero;
                uint4 w = w0;
                if (isA) {
                    if (kb == I) {
                        w.x &= keep_gt(r, 0); w.y &= keep_gt(r, 1); w.z &= keep_gt(r, 2); w.w &= keep_gt(r, 3);
                    }
                } else if (kb >= 2 * J) {
                    const int lim = r - 128 * (kb - 2 * J);
                    w.x &= keep_lt(lim, 0); w.y &= keep_lt(lim, 1); w.z &= keep_lt(lim, 2); w.w &= keep_lt(lim, 3);
                }
                mbar_wait(empty0 + 8 * stage, sphase ^ 1);
                uint8_t* tile_smem = stage_base + stage * TC_STAGE_BYTES + (isA ? 0 : TC_A_BYTES);
                unpack_row_to_smem(tile_smem, r, w);
                fence_proxy_async_smem();
                mbar_arrive(full0 + 8 * stage);
                if (++stage == TC_STAGES) { stage = 0; sphase ^= 1; }
                w0 = w1; w1 = w2;
            }

            // ---- epilogue: TMEM -> registers -> mask by R[i][j], i<j -> histogram
            mbar_wait(tmem_full, tphase);
            tphase ^= 1;
            tc_fence_after();
            const long long i = i0 + 32 * q4 + lane;
            const uint32_t* relrow32 = reinterpret_cast<const uint32_t*>(rel + (i < N ? i : 0) * stride_words);
            for (int c = c_begin; c < c_end; ++c) {
                uint32_t v[32];
                tmem_ld_32x32(tmem_base + ((uint32_t)(32 * q4) << 16) + (uint32_t)(32 * c), v);
                const long long jc = j0 + 32 * c;
                uint32_t relw = (i < N) ? __ldg(relrow32 + (jc >> 5)) : 0u;
                // keep only columns j > i
                if (jc + 31 <= i) relw = 0u;
                else if (jc <= i) relw &= 0xFFFFFFFFu << (int)(i - jc + 1);
#pragma unroll
                for (int x = 0; x < 32; ++x) {
                    const int n = (int)v[x];
                    if (((relw >> x) & 1u) && n <= kmax) {
                        if (n < TC_HIST) atomicAdd(&hist[n], 1u);
                        else atomicAdd(&counts[n], 1ULL);
                    }
                }
            }
            tc_fence_before();
            mbar_arrive(tmem_empty);
        }
    } else {
        // ================================================================== MMA issuer (one warp, lane 0 issues)
        uint32_t stage = 0, sphase = 0, ephase = 0;
        int done_tiles = 0;
        for (int rd = 0; rd < rounds; ++rd) {
            const int t = rd * G + ((rd & 1) ? (G - 1 - cta) : cta);
            if (t >= ntiles) continue;
            const int2 tile = tiles[t];
            const int kb_begin = tile.x, kb_end = 2 * tile.y + 2;
            if (done_tiles > 0) {                       // accumulator must have been drained
                mbar_wait(tmem_empty, ephase);
                ephase ^= 1;
            }
            tc_fence_after();
            for (int kb = kb_begin; kb < kb_end; ++kb) {
                mbar_wait(full0 + 8 * stage, sphase);
                tc_fence_after();
                if (lane == 0) {
                    const uint32_t a_addr = smem_u32(stage_base + stage * TC_STAGE_BYTES);
                    const uint64_t adesc = make_kmajor_sw128_desc(a_addr);
                    const uint64_t bdesc = make_kmajor_sw128_desc(a_addr + TC_A_BYTES);
#pragma unroll
                    for (int kk = 0; kk < TC_KS / 32; ++kk)   // K = 32 bytes per instruction: +2 in 16-byte units
                        umma_i8(tmem_base, adesc + 2 * kk, bdesc + 2 * kk, TC_IDESC, (kb > kb_begin || kk > 0) ? 1u : 0u);
                    umma_commit(empty0 + 8 * stage);
                    if (kb == kb_end - 1) umma_commit(tmem_full);
                }
                __syncwarp();
                if (++stage == TC_STAGES) { stage = 0; sphase ^= 1; }
            }
            ++done_tiles;
        }
    }

    // ---- teardown: flush the privatised histogram, release TMEM
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    for (int b = tid; b < TC_HIST && b <= kmax; b += TC_THREADS)
        if (hist[b]) atomicAdd(&counts[b], (unsigned long long)hist[b]);
    if (warp == TC_PRODUCER_WARPS) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(TC_TMEM_COLS)
                     : "memory");
    }
}

}  // namespace csg
