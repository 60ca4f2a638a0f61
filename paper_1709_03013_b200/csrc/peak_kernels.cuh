// Measurement aids (csg_measure_peak): the roofline denominators of the two interval-kernel variants, measured on
// the device the library runs on instead of derived from data-sheet numbers.
//
//   tensor_peak_kernel<KIND>: what the tensor cores sustain on exactly the instruction the interval kernel issues
//     (tcgen05.mma.cta_group::2, M = N = 256, K = 64 e2m1 with block32 scales and A in TMEM, or K = 32 u8 with both
//     operands in shared memory), with NO producers, no TMA, no epilogue: one thread per CTA pair issues MMAs back to
//     back over a ring of operand slots that were filled once.  Operands are pseudo-random relation bits expanded
//     the same way the interval kernel expands them (a tensor core fed zeros draws less power and clocks higher).
//   alu_peak_kernel<MODE>: issue rate of the bitset variant's inner instruction mix (LOP3 AND + POPC + IADD per 32
//     bit-tests, PAPER.md:323-387 restated for the integer pipes) and of POPC / LOP3 alone.
//
// Nothing here is on the hot path.
#pragma once
#include "tensor_kernel.cuh"

namespace csg {

__device__ __forceinline__ uint32_t peak_hash(uint32_t x) {
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

// groups: number of 4-MMA groups (one "stage" of the interval kernel each) issued per cluster.
template <int KIND>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(TC_THREADS, 1)
tensor_peak_kernel(int groups, unsigned int* __restrict__ sink) {
    using T = TcTraits<KIND>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem = smem_raw + (smem0 - smem_u32(smem_raw));
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + T::OFF_BARS + 8 * T::NUM_BARS);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = cluster_ctarank();
    const uint32_t bar0 = smem0 + T::OFF_BARS;                  // one barrier per ring slot + a final one
    const uint32_t bar_done = bar0 + 8 * T::STAGES;
    if (tid == 0) {
        for (int s = 0; s <= T::STAGES; ++s) mbar_init(bar0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == TC_MMA_WARP) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                     "n"(T::TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    // operand slots: expanded pseudo-random relation bits (density 1/2), same encodings as the interval kernel
    uint32_t* words = reinterpret_cast<uint32_t*>(smem);
    for (int x = tid; x < T::STAGES * T::STAGE_BYTES / 4; x += TC_THREADS) {
        const uint32_t h = peak_hash(x * 2654435761u + 97u * blockIdx.x);
        const int cls = (x >> 2) & 3;                           // chunk = class, as unpack_group_fp4 lays them out
        words[x] = KIND == KIND_FP4 ? (h & (0x11111111u << (cls == 3 ? 2 : cls))) : (h & 0x80808080u);
    }
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    if (KIND == KIND_FP4 && warp < 4) {
        tmem_fill_32x32(tmem_base + ((uint32_t)(32 * warp) << 16) + T::TMEM_SF, TC_SF_CELL);
        for (int s = 0; s < T::STAGES; ++s) {                   // the A ring in TMEM
            uint4 o[8];
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const uint32_t h = peak_hash(tid * 64 + s * 8 + m + 1234567u);
                o[m] = make_uint4(h & (0x11111111u << (m % 3)), peak_hash(h) & (0x11111111u << (m % 3)),
                                  peak_hash(h + 1) & (0x11111111u << (m % 3)), peak_hash(h + 2) & (0x11111111u << (m % 3)));
            }
            tmem_st_32x32(tmem_base + ((uint32_t)(32 * warp) << 16) + T::TMEM_A + 32u * s, o);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        tc_fence_before();
    }
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();

    if (warp == TC_MMA_WARP && rank == 0) {
        const bool issuer = elect_one();
        uint32_t slot = 0, parity = 0;
        const uint64_t adesc0 = make_kmajor_sw128_desc(smem0), bdesc0 = make_kmajor_sw128_desc(smem0 + T::OFF_B);
        for (int g = 0; g < groups; ++g) {
            if (g >= T::STAGES) mbar_wait(bar0 + 8 * slot, parity);   // the group that used this slot last has completed
            if (issuer) {
                const uint64_t soff = (uint64_t)(slot * (T::STAGE_BYTES >> 4));
#pragma unroll
                for (int kk = 0; kk < TC_ROW_BYTES / 32; ++kk) {
                    const uint32_t acc = (g > 0 || kk > 0) ? 1u : 0u;
                    if (KIND == KIND_FP4)
                        umma_mxf4_2cta_ts(tmem_base, tmem_base + T::TMEM_A + 32u * slot + 8u * kk, bdesc0 + soff + 2 * kk,
                                          (kk & 1) ? TC_IDESC_FP4_ODD : TC_IDESC_FP4, acc, tmem_base + T::TMEM_SF,
                                          tmem_base + T::TMEM_SFB);
                    else
                        umma_i8_2cta(tmem_base, adesc0 + soff + 2 * kk, bdesc0 + soff + 2 * kk, TC_IDESC, acc);
                }
                umma_commit_2cta(bar0 + 8 * slot);
            }
            if (++slot == (uint32_t)T::STAGES) { slot = 0; if (g >= T::STAGES) parity ^= 1; }
        }
        if (issuer) umma_commit_2cta(bar_done);
    }
    mbar_wait(bar_done, 0);                                      // both CTAs: every MMA has completed
    tc_fence_after();
    if (warp == 0) {                                             // keep the accumulators observable
        uint32_t v[32];
        tmem_ld_32x32(tmem_base, v);
        if (v[lane] == 0x12345u) sink[0] = v[0];
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    if (warp == TC_MMA_WARP)
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(T::TMEM_COLS) : "memory");
}

// MODE 0: the bitset variant's mix, per step 1 LOP3 (and) + 1 POPC + 1 IADD on 8 independent chains per thread;
// MODE 1: POPC only; MODE 2: LOP3 only.  Each thread executes iters x 8 steps.
constexpr int ALU_PEAK_THREADS = 256;
template <int MODE>
__global__ void __launch_bounds__(ALU_PEAK_THREADS, 4) alu_peak_kernel(int iters, unsigned int* __restrict__ sink) {
    uint32_t a[8], acc[8];
    const uint32_t seed = blockIdx.x * ALU_PEAK_THREADS + threadIdx.x;
#pragma unroll
    for (int c = 0; c < 8; ++c) { a[c] = peak_hash(seed * 8 + c); acc[c] = c; }
    uint32_t b = peak_hash(seed ^ 0xabcdefu);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            if (MODE == 0) {
                uint32_t t, p;
                asm volatile("and.b32 %0, %1, %2;" : "=r"(t) : "r"(a[c]), "r"(b));
                asm volatile("popc.b32 %0, %1;" : "=r"(p) : "r"(t));
                asm volatile("add.u32 %0, %0, %1;" : "+r"(acc[c]) : "r"(p));
            } else if (MODE == 1) {
                asm volatile("popc.b32 %0, %0;" : "+r"(acc[c]));
            } else {
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(acc[c]) : "r"(a[c]), "r"(b));
            }
        }
        b += 0x9e3779b9u;
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < 8; ++c) r ^= acc[c];
    if (r == 0x7654321u) sink[0] = r;
}

}  // namespace csg
