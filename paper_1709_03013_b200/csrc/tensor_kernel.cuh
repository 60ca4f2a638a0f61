// Tensor-core variant of the interval kernel: a tiled binary "GEMM" on tcgen05 (sm_100a), CTA pairs.
//
// What it computes (Sec. 4.1, Fig. 2, Alg. 5 l.7): for every related
// pair i<j, n_ij = sum_{i<k<j} R[i][k] * R[j][k], bucketed into counts[n_ij].  With U[i][k] = R[i][k]*[k>i]
// and L[j][k] = R[j][k]*[k<j] this is the matrix product C = U * L^T restricted to the upper triangle and
// masked by R[i][j] -- a dense contraction over k, so it runs on the 5th-generation tensor cores:
//
//   * a cluster of two CTAs (one SM pair) owns a 256 x 256 tile of pairs (rows i of block I, rows j of block J)
//     and sweeps K from the first column of block I to the last column of block J in stages of 128 (int8 kind)
//     or 256 (fp4 kind) columns.  CTA rank p holds rows i0+128p.. of the A operand and rows j0+128p.. of the B
//     operand, so each SM expands 256 rows per stage for a 256 x 256 x stage product, and each tensor core reads
//     half of B from its own shared memory and half from its peer's;
//   * per CTA one TMA thread streams the packed bits of its 256 rows (one copy = a group of 2 stages per row,
//     32- or 64-byte-swizzled 2D boxes of 128 rows) into a 4-deep shared-memory ring: whole sectors, one issuing
//     thread; rows >= N and columns beyond the row are zero-filled by the TMA unit;
//   * 16 producer warps in two sets of 8, one row per thread.  Set p expands both stages of every second group
//     (TC_WHOLE_GROUP; the older split "set p takes stage p of every group" remains as a compile-time option):
//     LDS.128 of the row's bits -> open-range mask where needed -> shifts/ANDs -> operand tile.  The B tile is a
//     K-major, 128-byte-swizzled shared-memory tile (UMMA canonical layout); the A tile is the same for the int8
//     kind and lives in TMEM for the fp4 kind (tcgen05.st, lane = row; see TcTraits).  The order of the k's
//     inside a 32-bit word is permuted identically for both operands; the MMA sums over k, so nothing changes.
//     The packed-bit buffer goes back to the TMA thread only after the stores that consume its words (see the
//     comment in the stage loop: an arrive placed right after the LDS instructions was a race);
//   * one thread of the leader CTA issues tcgen05.mma.cta_group::2 four times per stage (kind::i8: u8 x u8 -> s32;
//     kind::mxf4 with unit block scales: e2m1 x e2m1 -> f32 holding exact integers); each CTA's 128 accumulator
//     rows live in 256 columns of its own TMEM; tcgen05.commit (multicast) hands the stage back to the producers
//     of both CTAs.  Operand ring: 4 stages (int8), 6 stages (fp4);
//   * the open range i<k<j costs nothing in the steady state: only the stages that overlap block I need the k>i
//     mask and only those that overlap block J the k<j mask;
//   * fused epilogue by the producer warps: tcgen05.ld of their CTA's accumulators, bit R[i][j] (and i<j), n_ij
//     into a privatised shared-memory histogram (the launch's hist_bins) or straight into the global counts (higher bins,
//     smeared action only).  The first two groups of the NEXT tile are expanded before the epilogue of a tile, so
//     the tensor cores restart as soon as the accumulators are drained.  No N x N count matrix ever reaches HBM.
//
// Template FLAGS select what else is compiled in, so that a launch pays only for what it uses: TCF_WAIT (drift
// throttle: the TMA thread may wait for the finished-tile counter before it starts a tile), TCF_GATE (host-copy gate of
// csg_action_host: tiles wait for the chunks of the matrix they read; implies the throttle code), TCF_SPARSE
// (block-sparse K sweep: the roles walk the live-group masks of the occupancy map instead of a counted loop; fp4
// kind), TCF_BATCH (csg_action_batch: tiles of many sets in one launch), TCF_DUMP (test hook csg_tile_interval_sizes: the epilogue writes every n_ij of the listed tiles instead of
// bucketing it), TCF_ABLATE (only in the separate -DCSG_ABLATE build of paper_1709_03013_b200/ablate.py, never in
// libcsg.so).
// `dbg` (csg_set_debug of the ABLATE build; 0 and compiled out everywhere else) switches parts of the kernel off
// for timing ablations (1: no MMA issue, 2: no
// expansion arithmetic, 4: no operand stores, 8: no bucketing in the epilogue, 16: no fence before publishing a stage, 32: no
// packed-bit ring, 64: producers free-running with no MMA thread and no epilogue, 128: no prefill of the next tile
// before an epilogue, 256: no open-range masks); any non-zero value gives wrong counts.
//
// Tiles come from a host-built list (csg.cu: build_tile_schedule: deepest first, for large matrices in L2-sized
// patches) and are dealt in boustrophedon order over the persistent clusters (one per SM pair), which balances
// the triangular workload without a global counter.
#pragma once
#include <cuda.h>

#include <cstdint>

namespace csg {

constexpr int TC_T = 256;                  // tile edge in pairs (UMMA M = N = 256 over the CTA pair)
constexpr int TC_SET_SHIFT = 14;           // tiles[t].x = I | set << 14: which causal set of a batch the tile belongs to (csg_action_batch)
constexpr int TC_ROWS_A = 128;             // A rows per CTA
constexpr int TC_ROWS_B = 128;             // B rows per CTA
constexpr int TC_ROWS = TC_ROWS_A + TC_ROWS_B;
constexpr int TC_ROW_BYTES = 128;          // bytes per operand row per stage in smem (one 128-byte swizzle row)
constexpr int TC_A_BYTES = TC_ROWS_A * TC_ROW_BYTES;  // 16 KiB
constexpr int TC_B_BYTES = TC_ROWS_B * TC_ROW_BYTES;  // 16 KiB
constexpr int TC_GROUP = 2;                // stages covered by one packed-bit copy
constexpr int TC_BITS_BOX_ROWS = 128;
constexpr int TC_PRODUCER_WARPS = 16;      // two sets of 8 warps; in a set: 4 warps for the A rows, 4 for the B rows
constexpr int TC_PRODUCERS = TC_PRODUCER_WARPS * 32;
constexpr int TC_MMA_WARP = TC_PRODUCER_WARPS;
constexpr int TC_TMA_WARP = TC_PRODUCER_WARPS + 1;
constexpr int TC_THREADS = TC_PRODUCERS + 64;  // + the MMA warp + the TMA warp
#ifndef CSG_WHOLE_GROUP
#define CSG_WHOLE_GROUP 1
#endif
#ifndef CSG_SCALE_CLASSES
#define CSG_SCALE_CLASSES 1                // fp4 operands: position classes keep their nibble bit, block scales undo it (unpack_group_fp4)
#endif
constexpr bool TC_WHOLE_GROUP = CSG_WHOLE_GROUP != 0;   // a producer set expands both stages of every second group
constexpr int TC_MAX_LEAD = 1;                 // rounds a cluster may run ahead of the average (L2 sharing inside a patch)
constexpr int TC_THROTTLE_MAX_POLLS = 1 << 15; // polls of >= 200 ns in ONE wait before a cluster stops throttling for good (see the TMA warp)
constexpr int TCF_ABLATE = 1, TCF_WAIT = 2, TCF_DUMP = 4, TCF_GATE = 8, TCF_SPARSE = 16, TCF_BATCH = 32;   // template FLAGS of tensor_action_kernel
#ifndef CSG_PREFILL_GROUPS
#define CSG_PREFILL_GROUPS 2
#endif
#ifndef CSG_BITS_BUFS
#define CSG_BITS_BUFS 4
#endif
#ifndef CSG_STATIC_DBG
#define CSG_STATIC_DBG 0                   // measurement builds only (ablate.py --static): the dbg switches as a compile-time constant
#endif
constexpr int TC_PREFILL_GROUPS = CSG_PREFILL_GROUPS;   // groups (2 stages each) of the next tile expanded before a tile's epilogue
// Privatised low bins per CTA (u32, shared memory, the last region of the dynamic window; the launch says how many).
// Higher bins -- whole-histogram launches (smeared action) only -- go to the global histogram with one red.add per
// value, and scattered global atomics run at 185 G/s on the device (1.57 clk each per SM, measured; u32 and u64
// alike): a 2D set at N = 262144 sends 1.5e10 of them, 8 % of the launch.  In a 2D order the share of related pairs with
// n_ij < B is about 4x(-ln x - 1), x = B/N: 12 % at B = 2048, 39 % at B = 12288 (48 KiB: what is left of the 227 KiB
// beside the operand ring).  Measured: config 4 835.6 -> 819.6 ms, config 5 94.1 -> 92.4 ms with 12288 bins -- but
// config 3, whose epilogue needs four bins, 81.8 -> 83.5 ms (too little L1 is left beside 213 KiB of shared memory).  So
// the host gives 12288 bins to launches that can reach bins >= 2048 and 2048 to all others.
constexpr int TC_HIST = 2048;              // every launch has at least these
constexpr int TC_HIST_WHOLE = 12288;       // launches with kmax >= TC_HIST

// The two operand encodings of the kernel.
//   KIND_I8 : one relation bit -> one u8 (0 or 1 << TB); tcgen05.mma kind::i8, K = 32 per instruction, s32
//             accumulators; a stage row of 128 bytes covers 128 columns.
//   KIND_FP4: one relation bit -> one e2m1 nibble, two per byte; tcgen05.mma kind::mxf4 (block32 UE8M0 scales),
//             K = 64 per instruction, f32 accumulators holding 4 n_ij (exact below 2^24); a stage row of 128 bytes
//             covers 256 columns, at twice the int8 MAC rate.  The nibble of a set bit is 0.5, 1.0, 2.0 or 2.0
//             depending on the bit's position class inside its 32-bit word, and the block scales (4, 2, 1, 1) undo
//             that, so every product of two set bits is 4 (see unpack_group_fp4).
constexpr int KIND_I8 = 0, KIND_FP4 = 1;
template <int KIND>
struct TcTraits {
    static constexpr int STAGE_COLS = KIND == KIND_FP4 ? 256 : 128;           // k columns per stage
    static constexpr int WORDS = STAGE_COLS / 32;                             // packed 32-bit words per row per stage
    static constexpr int BITS_ROW_BYTES = TC_GROUP * STAGE_COLS / 8;          // 32 or 64 bytes per row per copy
    static constexpr int BITS_BOX_BYTES = TC_BITS_BOX_ROWS * BITS_ROW_BYTES;
    static constexpr int BITS_BUF_BYTES = TC_ROWS * BITS_ROW_BYTES;           // 8 or 16 KiB
    // fp4 keeps only the B operand in shared memory (A lives in TMEM, see A_TMEM).
#ifndef CSG_A_IN_TMEM
#define CSG_A_IN_TMEM 1
#endif
    static constexpr bool A_IN_TMEM = KIND == KIND_FP4 && CSG_A_IN_TMEM;
    static constexpr int OFF_B = A_IN_TMEM ? 0 : TC_A_BYTES;                  // B tile inside a stage
    static constexpr int STAGE_BYTES = OFF_B + TC_B_BYTES;                    // 16 or 32 KiB
    // Ring of operand stages (even: the two producer sets own alternate slots).  The round trip of a slot
    // (producers arrive on `full` in the leader CTA -> MMA thread -> tcgen05.commit multicast -> `empty`) measured
    // ~1400 clk with everything else switched off, so 4 slots cap the pace at one stage per ~340 clk before any
    // work is done; fp4 has room for 6 (B only in shared memory, A ring = 6 x 32 TMEM columns).
    static constexpr int STAGES = A_IN_TMEM ? 6 : 4;
    static constexpr int BITS_BUFS = CSG_BITS_BUFS;
    static constexpr int NUM_BARS = 2 * STAGES + 2 + 2 * BITS_BUFS;
    static constexpr int OFF_BITS = STAGES * STAGE_BYTES;
    static constexpr int OFF_BARS = OFF_BITS + BITS_BUFS * BITS_BUF_BYTES;
    static constexpr int OFF_HIST = (OFF_BARS + 8 * NUM_BARS + 16 + 15) & ~15;  // after the barriers and the TMEM slot
    static constexpr int smem_bytes(int hist_bins) { return OFF_HIST + hist_bins * 4 + 1024; }   // + alignment slack
    static constexpr int SMEM_BYTES = smem_bytes(TC_HIST);
    static constexpr int TMEM_COLS = KIND == KIND_FP4 ? 512 : 256;            // fp4: + scale factors + the A ring
    // fp4: the A operand never touches shared memory.  The A producers write their expanded rows straight into
    // TMEM (lane = row, 32-bit column j of a K=64 slice = bytes 4j..4j+3 of the row's 32-byte slice, the same
    // order as the K-major shared-memory row; measured with a one-nibble-per-row probe) and the MMA reads A from
    // there: half of the operand stores and half of the tensor cores' operand reads leave the shared-memory pipe.
    static constexpr bool A_TMEM = A_IN_TMEM;
    static constexpr int TMEM_SF = 256;                                       // scale factors: SFA at +0, SFB at +16
    static constexpr int TMEM_SFB = TMEM_SF + 16;
    static constexpr int TMEM_A = 288;                                        // A ring: STAGES x 32 columns (288..479)
};

// ---------------------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// True in exactly one lane of a converged warp.  ptxas knows that a branch on this predicate has a single active
// thread, so the tcgen05 / TMA instructions inside it are issued directly; inside `if (lane == 0)` it wraps every
// one of them in an ELECT / BRA.U.ANY loop over the "possibly several" active lanes (5 extra instructions each).
__device__ __forceinline__ bool elect_one() {
    uint32_t is_elected;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(is_elected));
    return is_elected != 0;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_cta(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Arrive on a barrier of any CTA of the cluster (address from map_to_cta).  Default semantics on purpose: the
// operand bytes reach the tensor cores through the async proxy, ordered by fence.proxy.async before this arrive;
// a .release.cluster here compiles to MEMBAR.ALL.GPU + an L1 invalidate per stage and tripled the stage time.
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_bar) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@!p bra WAIT_%=;\n\t}" ::"r"(bar), "r"(parity) : "memory");   // one branch, not taken when the phase is complete
}
// One non-blocking probe of the barrier phase; lets the caller overlap the probe latency with other work.
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// 2D tiled TMA load global -> shared; completes bytes on `bar`.  c0 = byte column, c1 = row.
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr)
                 : "memory");
    return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint4& v) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w)
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// Same fence, placed AFTER the computation of the 32 registers it names: the fake register dependency stops the
// compiler from sinking the unpack arithmetic below the fence, so the fence finds the previous stage's stores
// already drained.
__device__ __forceinline__ void fence_proxy_async_smem_after(uint4 (&o)[8]) {
    asm volatile("fence.proxy.async.shared::cta;"
                 : "+r"(o[0].x), "+r"(o[0].y), "+r"(o[0].z), "+r"(o[0].w), "+r"(o[1].x), "+r"(o[1].y), "+r"(o[1].z),
                   "+r"(o[1].w), "+r"(o[2].x), "+r"(o[2].y), "+r"(o[2].z), "+r"(o[2].w), "+r"(o[3].x), "+r"(o[3].y),
                   "+r"(o[3].z), "+r"(o[3].w), "+r"(o[4].x), "+r"(o[4].y), "+r"(o[4].z), "+r"(o[4].w), "+r"(o[5].x),
                   "+r"(o[5].y), "+r"(o[5].z), "+r"(o[5].w), "+r"(o[6].x), "+r"(o[6].y), "+r"(o[6].z), "+r"(o[6].w),
                   "+r"(o[7].x), "+r"(o[7].y), "+r"(o[7].z), "+r"(o[7].w)
                 :
                 : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// D[tmem] (+)= A[smem] * B[smem]^T, u8 x u8 -> s32, over the CTA pair (issued by the leader CTA only).
__device__ __forceinline__ void umma_i8_2cta(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                             uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d), "l"(adesc), "l"(bdesc),
        "r"(idesc), "r"(accumulate) : "memory");
}
// Arrive on the barrier at this shared-memory offset in BOTH CTAs once all tcgen05 ops issued so far completed.
__device__ __forceinline__ void umma_commit_2cta(uint32_t bar) {
    asm volatile(
        "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
        "h"((uint16_t)3) : "memory");
}
// 32 lanes x 32 consecutive 32-bit columns: thread t of the warp gets lane (base+t), columns c..c+31.
__device__ __forceinline__ void tmem_ld_32x32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n\t"
        "tcgen05.wait::ld.sync.aligned;"   // same asm statement: nothing that reads v[] can be scheduled above the wait
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]),
          "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]),
          "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]),
          "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}

// Shared-memory matrix descriptor: K-major operand, 128-byte swizzle, rows of 128 bytes, 8-row groups
// 1024 bytes apart (SBO), descriptor version 1 (sm_100).
__device__ __forceinline__ uint64_t make_kmajor_sw128_desc(uint32_t smem_addr) {
    const uint32_t lo = ((smem_addr >> 4) & 0x3FFFu) | (1u << 16);           // start address, LBO = 1 (unused)
    const uint32_t hi = (1024u >> 4) | (1u << 14) | (2u << 29);              // SBO, version, SWIZZLE_128B
    return (static_cast<uint64_t>(hi) << 32) | lo;
}
// Instruction descriptor, kind::i8: D = s32, A = B = u8, both K-major, N = 256, M = 256 (cta_group::2).
constexpr uint32_t TC_IDESC = (2u << 4) | ((256u >> 3) << 17) | ((256u >> 4) << 24);

// D[tmem] (+)= A[smem] * B[smem]^T, e2m1 x e2m1 -> f32 with UE8M0 block scales (one per 32 k) read from TMEM,
// over the CTA pair (issued by the leader CTA only).  K = 64 per instruction.
__device__ __forceinline__ void umma_mxf4_2cta(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                               uint32_t accumulate, uint32_t tmem_sfa, uint32_t tmem_sfb) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::mxf4.block_scale.block32 [%0], %1, %2, %3, [%5], [%6], p;\n\t}" ::"r"(tmem_d),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(tmem_sfa), "r"(tmem_sfb) : "memory");
}
// Instruction descriptor, kind::mxf4 block scaled: A = B = e2m1 (1), scales UE8M0 (1), K-major, N = 256, M = 256,
// scale-factor ids 0, K = 64.
constexpr uint32_t TC_IDESC_FP4 = (1u << 7) | (1u << 10) | ((256u >> 3) << 17) | (1u << 23) | ((256u >> 4) << 24);
// the same with scale-factor ids 2 for both operands (bits 4-5: B, bits 29-30: A): the two scales of the
// instruction's two 32-k blocks are bytes 2, 3 of the 32-bit scale cell instead of bytes 0, 1
constexpr uint32_t TC_IDESC_FP4_ODD = TC_IDESC_FP4 | (CSG_SCALE_CLASSES ? ((2u << 4) | (2u << 29)) : 0u);
// 32 lanes x 32 columns store of one value (fills the scale-factor region of TMEM).
__device__ __forceinline__ void tmem_fill_32x32(uint32_t taddr, uint32_t v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, "
        "%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1};" ::"r"(taddr), "r"(v) : "memory");
}

// 32 lanes x 32 columns: thread t of the warp writes its 32 registers (8 x uint4) to lane (base+t), columns c..c+31.
__device__ __forceinline__ void tmem_st_32x32(uint32_t taddr, const uint4 (&o)[8]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
        "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(taddr),
        "r"(o[0].x), "r"(o[0].y), "r"(o[0].z), "r"(o[0].w), "r"(o[1].x), "r"(o[1].y), "r"(o[1].z), "r"(o[1].w),
        "r"(o[2].x), "r"(o[2].y), "r"(o[2].z), "r"(o[2].w), "r"(o[3].x), "r"(o[3].y), "r"(o[3].z), "r"(o[3].w),
        "r"(o[4].x), "r"(o[4].y), "r"(o[4].z), "r"(o[4].w), "r"(o[5].x), "r"(o[5].y), "r"(o[5].z), "r"(o[5].w),
        "r"(o[6].x), "r"(o[6].y), "r"(o[6].z), "r"(o[6].w), "r"(o[7].x), "r"(o[7].y), "r"(o[7].z), "r"(o[7].w)
        : "memory");
}
// Wait for this thread's tcgen05.st's, then order them before the mbarrier arrive that follows.  Like
// fence_proxy_async_smem_after, it names the registers of the NEXT stage so that their arithmetic stays above it.
__device__ __forceinline__ void tmem_wait_st_after(uint4 (&o)[8]) {
    asm volatile("tcgen05.wait::st.sync.aligned;\n\ttcgen05.fence::before_thread_sync;"
                 : "+r"(o[0].x), "+r"(o[0].y), "+r"(o[0].z), "+r"(o[0].w), "+r"(o[1].x), "+r"(o[1].y), "+r"(o[1].z),
                   "+r"(o[1].w), "+r"(o[2].x), "+r"(o[2].y), "+r"(o[2].z), "+r"(o[2].w), "+r"(o[3].x), "+r"(o[3].y),
                   "+r"(o[3].z), "+r"(o[3].w), "+r"(o[4].x), "+r"(o[4].y), "+r"(o[4].z), "+r"(o[4].w), "+r"(o[5].x),
                   "+r"(o[5].y), "+r"(o[5].z), "+r"(o[5].w), "+r"(o[6].x), "+r"(o[6].y), "+r"(o[6].z), "+r"(o[6].w),
                   "+r"(o[7].x), "+r"(o[7].y), "+r"(o[7].z), "+r"(o[7].w)
                 :
                 : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]^T, kind::mxf4 block scaled, over the CTA pair: each CTA's half of A sits at the
// same address of its own TMEM.
__device__ __forceinline__ void umma_mxf4_2cta_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc,
                                                  uint32_t accumulate, uint32_t tmem_sfa, uint32_t tmem_sfb) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::mxf4.block_scale.block32 [%0], [%1], %2, %3, [%5], [%6], p;\n\t}" ::"r"(tmem_d),
        "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(tmem_sfa), "r"(tmem_sfb) : "memory");
}

// ---------------------------------------------------------------------------------------------- bit expansion
// KIND_I8.  One 32-bit word of a row (32 k's) -> 32 operand bytes (two 16-byte chunks), each 0 or 1 << TB.
// Class q of the word = bits q, q+8, q+16, q+24; they go to bit TB of the four bytes of one 32-bit lane, so one
// shift and one AND expand four k's.  Left shifts (q < TB) may be issued as IMAD.SHL on the FMA pipe, which
// unloads the ALU pipe that carries the ANDs: TB = 7 needs no right shift at all.  The order of the k's inside
// the word is permuted; both operands use the same permutation and the MMA sums over k.
template <int TB>
__device__ __forceinline__ uint32_t unpack_class(uint32_t x, int q) {
    constexpr uint32_t M = 0x01010101u << TB;
    return (q < TB ? (x << (TB - q)) : (x >> (q - TB))) & M;
}
template <int TB>
__device__ __forceinline__ void unpack_word(uint32_t x, uint4& lo, uint4& hi) {
    lo.x = unpack_class<TB>(x, 0); lo.y = unpack_class<TB>(x, 1);
    lo.z = unpack_class<TB>(x, 2); lo.w = unpack_class<TB>(x, 3);
    hi.x = unpack_class<TB>(x, 4); hi.y = unpack_class<TB>(x, 5);
    hi.z = unpack_class<TB>(x, 6); hi.w = unpack_class<TB>(x, 7);
}
// KIND_FP4.  Four 32-bit words (128 k's) -> four 16-byte chunks of 32 e2m1 nibbles each.  Class q of a word =
// its bits q, q+4, ..., q+28 = bit q of its eight nibbles.  Chunk q of the group holds class q of all four words,
// and a chunk is exactly one block of 32 k's with one UE8M0 scale, so a class may stay where it is:
//     class 0: x & 0x11111111 -> nibbles 0b0001 = 0.5,  block scale 4      class 2: x & 0x44444444 -> 0b0100 = 2.0, scale 1
//     class 1: x & 0x22222222 -> nibbles 0b0010 = 1.0,  block scale 2      class 3: (x >> 1) & 0x44444444 -> 2.0, scale 1
// (bit 3 of a nibble is the sign, so class 3 alone is shifted).  Both operands use the same encoding and the same
// scales, so every product of two set bits is (0.5*4)^2 = (1*2)^2 = (2*1)^2 = 4: the f32 accumulator holds 4 n_ij
// exactly.  5 ALU operations per word instead of the 7 of "every class shifted to bit 2, all scales 1".
// The MMA with even kk reads chunks 0, 1 (scale bytes 0, 1 of the TMEM cell), the one with odd kk chunks 2, 3
// (scale bytes 2, 3): TC_SF_CELL and the scale-factor ids of TC_IDESC_FP4_ODD.
constexpr uint32_t TC_SF_CELL = CSG_SCALE_CLASSES ? 0x7F7F8081u : 0x7F7F7F7Fu;   // UE8M0 bytes: 4, 2, 1, 1 (or all 1)
__device__ __forceinline__ void unpack_group_fp4(const uint32_t* w, uint4* o) {
#if CSG_SCALE_CLASSES
    o[0] = make_uint4(w[0] & 0x11111111u, w[1] & 0x11111111u, w[2] & 0x11111111u, w[3] & 0x11111111u);
    o[1] = make_uint4(w[0] & 0x22222222u, w[1] & 0x22222222u, w[2] & 0x22222222u, w[3] & 0x22222222u);
    o[2] = make_uint4(w[0] & 0x44444444u, w[1] & 0x44444444u, w[2] & 0x44444444u, w[3] & 0x44444444u);
    o[3] = make_uint4((w[0] >> 1) & 0x44444444u, (w[1] >> 1) & 0x44444444u, (w[2] >> 1) & 0x44444444u,
                      (w[3] >> 1) & 0x44444444u);
#else
#pragma unroll
    for (int m = 0; m < 4; ++m)
        o[m] = make_uint4((w[m] << 2) & 0x44444444u, (w[m] << 1) & 0x44444444u, w[m] & 0x44444444u,
                          (w[m] >> 1) & 0x44444444u);
#endif
}

// Word m (bits 32m..32m+31) of a stage: keep local bit positions p with p > r (operand U in the stages that
// hold row i's own column; r may be negative -> keep all, or beyond the stage -> keep none).
__device__ __forceinline__ uint32_t keep_gt(int r, int m) {
    const int s = r - 32 * m + 1;  // number of low bits to clear
    return s <= 0 ? 0xFFFFFFFFu : (s >= 32 ? 0u : (0xFFFFFFFFu << s));
}
// keep local bit positions p with p < lim (operand L in the stages that hold row j's own column)
__device__ __forceinline__ uint32_t keep_lt(int lim, int m) {
    const int s = lim - 32 * m;    // number of low bits to keep
    return s <= 0 ? 0u : (s >= 32 ? 0xFFFFFFFFu : ((1u << s) - 1u));
}

// K range of tile (I, J) in stages of COLS columns: from the stage holding column 256 I to the one holding
// column 256 J + 255, widened by one fully masked stage when the count would be odd (the two producer sets
// own the even and the odd ring slots).
template <int COLS>
__device__ __forceinline__ void tile_k_range(int I, int J, int& kb_begin, int& kb_end) {
    kb_begin = (256 * I) / COLS;
    kb_end = (256 * J + 255) / COLS + 1;
    if ((kb_end - kb_begin) & 1) {
        if (kb_begin > 0) --kb_begin; else ++kb_end;
    }
}

// Host-copy gate (csg_action_host): the matrix arrives in row chunks on a copy stream, which publishes the number of chunks
// delivered after each one (and after that chunk's rows of the occupancy map are complete); tile (I, J) reads the rows
// of blocks I and J only, and the host has worked out how many chunks that takes in its copy order.  The wait depends
// on the copy stream alone, never on another CTA.  The TMA thread waits before it fetches the tile's bits; with the
// block-sparse sweep the producers and the MMA thread wait, too, before they read the tile's occupancy rows (when the
// TMA thread is held up they catch up with it and would otherwise read rows that are not written yet).
__device__ __forceinline__ void wait_landed(const unsigned int* landed, unsigned int need, unsigned int& chunks_seen) {
    if (chunks_seen >= need) return;
    unsigned int got;
    while (true) {
        asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(got) : "l"(landed) : "memory");
        if (got >= need) break;
        __nanosleep(500);
    }
    chunks_seen = got;
}

// Live groups of a tile (block-sparse K sweep, template flag TCF_SPARSE).  A group = TC_GROUP = 2 consecutive stages, the
// unit of one packed-bit copy and of a producer set's turn.  occ = block occupancy of the relation matrix
// (occupancy_kernel.cuh; fp4 kind, 256-column stages, so stage kb of the sweep IS column block kb): stage kb of tile
// (I, J) multiplies block (I, kb) of U with block (J, kb) of L and is dead when either block is empty; a group is live
// when one of its two stages is.  live_groups_word returns the live mask of groups 32 gw .. 32 gw + 31 of the tile
// (group g = stages kb_begin + 2g, + 2g + 1); with occ == nullptr every group of the range is live.  All three roles of
// the kernel (TMA thread, producers, MMA thread) walk the same masks, so they agree on the sequence of groups without
// talking to each other.  Without TCF_SPARSE the sweep is the plain counted loop over all groups.
// Tried and dropped (measured at config 3, same box): an occupancy map in half-stages of 128 columns with the MMA thread
// skipping the dead half-stages inside live groups (6 % fewer MMAs): 83.7 ms against 81.8 -- the producers still expand
// them, they sit in the few groups at both ends of a sweep where the kernel is then producer-bound, and the longer
// issue loop costs every stage; running the dense configs through the mask loop with a null map: +4 % at config 1;
// one inlined call site for the epilogue through an end-of-tile call of the loop body: 87.6 ms (more loop state, spills);
// the MMA warp computing a tile's first mask word before it waits for the accumulators: no change (81.8 ms).
// COHERENT (TCF_GATE): the occupancy rows are written by another kernel WHILE this one runs (host-matrix pipeline: a
// row block is marked when its chunk has landed, before the chunk count that lets a tile start is published), so they
// are read from L2 (ld.relaxed.gpu) -- a row that shares a 128-byte line with one read earlier could otherwise come
// stale from L1.
template <bool COHERENT>
__device__ __forceinline__ uint32_t occ_load(const uint32_t* p) {
    if (!COHERENT) return __ldg(p);
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
template <bool COHERENT>
__device__ __forceinline__ uint32_t live_groups_word(const uint32_t* __restrict__ occI, const uint32_t* __restrict__ occJ,
                                                     int kb_begin, int kb_end, int gw) {
    const int rem = ((kb_end - kb_begin) >> 1) - 32 * gw;          // groups left from this word on
    const uint32_t in_range = rem >= 32 ? 0xFFFFFFFFu : ((1u << rem) - 1u);
    if (occI == nullptr) return in_range;
    const int s = kb_begin + 64 * gw;                              // first stage of the word
    const int w = s >> 5, sh = s & 31;
    const uint32_t a0 = occ_load<COHERENT>(occI + w) & occ_load<COHERENT>(occJ + w),
                   a1 = occ_load<COHERENT>(occI + w + 1) & occ_load<COHERENT>(occJ + w + 1),
                   a2 = occ_load<COHERENT>(occI + w + 2) & occ_load<COHERENT>(occJ + w + 2);  // rows end in zero words (OCC_PAD_WORDS)
    uint64_t S = ((uint64_t)__funnelshift_r(a1, a2, sh) << 32) | __funnelshift_r(a0, a1, sh);   // stages s .. s + 63
    S = (S | (S >> 1)) & 0x5555555555555555ull;                    // bit 2g: group g has a live stage
    S = (S | (S >> 1)) & 0x3333333333333333ull;                    // compress the even bits
    S = (S | (S >> 2)) & 0x0F0F0F0F0F0F0F0Full;
    S = (S | (S >> 4)) & 0x00FF00FF00FF00FFull;
    S = (S | (S >> 8)) & 0x0000FFFF0000FFFFull;
    S = (S | (S >> 16)) & 0x00000000FFFFFFFFull;
    return (uint32_t)S & in_range;
}
// Calls body(kb0) for the first stage kb0 of every live group of the tile, in ascending order; a tile without any
// live group still gets its first group (the MMA of a tile's first stage is what clears the accumulators).
template <bool SPARSE, bool COHERENT, class F>
__device__ __forceinline__ void for_live_groups(const uint32_t* __restrict__ occ, int occ_stride, int I, int J,
                                                int kb_begin, int kb_end, F&& body) {
    if (!SPARSE) {
        for (int kb0 = kb_begin; kb0 < kb_end; kb0 += TC_GROUP) body(kb0);
        return;
    }
    const uint32_t* occI = occ ? occ + (size_t)I * occ_stride : nullptr;
    const uint32_t* occJ = occ ? occ + (size_t)J * occ_stride : nullptr;
    const int nwords = (((kb_end - kb_begin) >> 1) + 31) >> 5;
    int done = 0;
    for (int gw = 0; gw <= nwords; ++gw) {
        uint32_t m = gw < nwords ? live_groups_word<COHERENT>(occI, occJ, kb_begin, kb_end, gw) : (done == 0 ? 1u : 0u);
        const int base = gw < nwords ? kb_begin + 64 * gw : kb_begin;
        while (m) {
            const int g = __ffs((int)m) - 1;
            m &= m - 1;
            ++done;
            body(base + 2 * g);
        }
    }
}

// KIND_I8: TB = bit of the operand byte that carries the relation bit: operands are 0 or 2^TB, every product is
// 4^TB, the accumulator holds n_ij << 2TB; the host picks the largest TB with (N-2) << 2TB < 2^31 (exact in s32).
// KIND_FP4: TB unused (pass 0); the f32 accumulator holds 4 n_ij, exact for n_ij < 2^22.
// tiles[t] = {I | set << TC_SET_SHIFT, J}: 256-row blocks, I <= J, of causal set `set` of a batch (0 for a single set).
// A batch (csg_action_batch) is `batch` matrices of N rows back to back: set b's row i is row b N + i of the TMA view
// and of `rel`, and its abundances go to counts + b * counts_stride with one global atomic per warp, bin and tile
// (template flag TCF_BATCH; without it: a single set, bins collected in the CTA's shared-memory histogram -- the
// decode and the second flush path cost 0.5 - 3 % when they were compiled into every instantiation).  The rows that a tile's
// 256-row blocks hold beyond N belong to the next set instead of being zero-filled; they only reach accumulators of
// rows i >= N, which the epilogue drops, and of columns j >= N, where row i's relation bits are zero padding.
// Grid = 2 x (number of SM pairs), cluster (2,1,1).
// hist_bins: bins of the CTA's private histogram (TC_HIST or TC_HIST_WHOLE; the launch's dynamic shared memory is
// TcTraits::smem_bytes(hist_bins)).
// progress (TCF_WAIT or TCF_GATE, may be NULL): zeroed counter of finished tiles, the drift throttle.  landed / tile_need (TCF_GATE,
// may be NULL): the host-copy gate -- *landed = number of row chunks of `rel` the copy stream has delivered so far,
// tile_need[t] = how many must be there before tile t may start.  dump (TCF_DUMP): ntiles x 256 x 256 int32, n_ij or -1.
template <int KIND, int TB, int FLAGS = 0>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(TC_THREADS, 1)
tensor_action_kernel(const __grid_constant__ CUtensorMap bits_map, const uint64_t* __restrict__ rel, long long N,
                     long long stride_words, int kmax, unsigned long long* __restrict__ counts,
                     const int2* __restrict__ tiles, int ntiles, int dbg_arg, unsigned int* __restrict__ progress_arg,
                     const unsigned int* __restrict__ landed_arg, const int* __restrict__ tile_need,
                     int* __restrict__ dump, const uint32_t* __restrict__ occ_arg, int occ_stride, int counts_stride,
                     int hist_bins) {
    constexpr bool ABLATE = (FLAGS & TCF_ABLATE) != 0, DUMP = (FLAGS & TCF_DUMP) != 0, GATE = (FLAGS & TCF_GATE) != 0;
    constexpr bool WAITS = (FLAGS & (TCF_WAIT | TCF_GATE)) != 0;        // the TMA thread may wait on global words
    constexpr bool SPARSE = (FLAGS & TCF_SPARSE) != 0 && KIND == KIND_FP4;   // block-sparse sweep: fp4 kind only (stage = column block)
    constexpr bool BATCH = (FLAGS & TCF_BATCH) != 0;                    // tiles carry a set index (csg_action_batch)
    constexpr int TILE_I_MASK = BATCH ? (1 << TC_SET_SHIFT) - 1 : -1;   // single set: tiles[t].x is the block index itself
    unsigned int* const progress = WAITS ? progress_arg : nullptr;      // compiled out of the instantiations that never wait
    const unsigned int* const landed = GATE ? landed_arg : nullptr;
    const uint32_t* const occ = SPARSE ? occ_arg : nullptr;
    using T = TcTraits<KIND>;
    // 0 and compiled out of every instantiation of libcsg.so.  Two measurement builds exist (paper_1709_03013_b200/ablate.py):
    // -DCSG_ABLATE (run-time switches through csg_set_debug; the tests in the hot loops make that build 28 % slower than the
    // product) and -DCSG_STATIC_DBG=<bits> (the same switches as a compile-time constant: what is left runs at product speed).
    const int dbg = CSG_STATIC_DBG != 0 ? CSG_STATIC_DBG : (ABLATE ? dbg_arg : 0);
    constexpr int COLS = T::STAGE_COLS, WORDS = T::WORDS;
    extern __shared__ uint8_t smem_raw[];
    // the dynamic shared window starts at the same offset in both CTAs, so this rounding is identical in both
    const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem = smem_raw + (smem0 - smem_u32(smem_raw));
    unsigned int* hist = reinterpret_cast<unsigned int*>(smem + T::OFF_HIST);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + T::OFF_BARS + 8 * T::NUM_BARS);

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = cluster_ctarank();          // 0 = leader (issues the MMAs)
    const uint32_t full0 = smem0 + T::OFF_BARS, empty0 = full0 + 8 * T::STAGES;
    const uint32_t tmem_full = empty0 + 8 * T::STAGES, tmem_empty = tmem_full + 8;
    const uint32_t bits_full0 = tmem_empty + 8, bits_empty0 = bits_full0 + 8 * T::BITS_BUFS;

    for (int b = tid; b < hist_bins; b += TC_THREADS) hist[b] = 0u;
    if (tid == 0) {
        for (int s = 0; s < T::STAGES; ++s) {
            mbar_init(full0 + 8 * s, TC_PRODUCER_WARPS);       // leader's copy is used: 8 warps of one producer set x 2 CTAs
            mbar_init(empty0 + 8 * s, 1);                      // multicast tcgen05.commit
        }
        mbar_init(tmem_full, 1);                               // multicast tcgen05.commit
        mbar_init(tmem_empty, 2 * TC_PRODUCER_WARPS);          // leader's copy is used
        for (int b = 0; b < T::BITS_BUFS; ++b) {
            mbar_init(bits_full0 + 8 * b, 1);                  // expect_tx arrive of the TMA thread
            mbar_init(bits_empty0 + 8 * b, TC_WHOLE_GROUP ? TC_PRODUCER_WARPS / 2 : TC_PRODUCER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == TC_MMA_WARP) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                     "n"(T::TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    if (KIND == KIND_FP4 && warp < 4) {
        // block scales: every 32-bit cell of TMEM columns 256..287 (all 128 lanes) holds the same four UE8M0 bytes,
        // so the row a cell belongs to does not matter: byte b scales the b-th chunk of a 64-byte operand group
        tmem_fill_32x32(tmem_base + ((uint32_t)(32 * warp) << 16) + T::TMEM_SF, TC_SF_CELL);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        tc_fence_before();
    }
    __syncthreads();
    cluster_sync_all();                               // both CTAs' barriers and scale factors are ready
    tc_fence_after();

    const int G = gridDim.x >> 1, cl = blockIdx.x >> 1;   // persistent clusters
    const int rounds = (ntiles + G - 1) / G;

    if (warp < TC_PRODUCER_WARPS) {
        // ================================================================== producers + epilogue
        // Two producer sets of 8 warps, one row per thread.  TC_WHOLE_GROUP (default): set p expands both stages of
        // every second 2-stage group (one buffer wait, one release and one trip through the loop per two stages);
        // otherwise set p expands stage p of every group.  Either way a warp has two stage times for the serial
        // chain wait -> expand -> fence -> arrive -> store of a stage.
        const int pset = warp >> 3;                   // 0 or 1: which stage of each group this thread expands
        const int prow = tid & 255;                   // row 0..255 of this CTA's staged rows
        const bool isA = prow < TC_ROWS_A;
        const int r = isA ? prow : prow - TC_ROWS_A;  // row inside this CTA's A or B operand tile
        const int rt = (int)rank * 128 + r;           // row inside the 256-row block of the cluster tile
        uint32_t sl = 0, sphase = 0;                  // this set's slot counter: operand slot = pset + 2*sl, and its parity
        uint32_t gsel = 0, slot0 = 0, spar = 0;       // TC_WHOLE_GROUP: running group count, first slot of the group, use parity
        uint32_t bb = 0, bphase = 0;                  // packed-bit ring position / parity
        int pending = -1;                             // ring stage written but not yet published
        const uint32_t row_smem = smem0 + (isA ? 0 : T::OFF_B) + (r >> 3) * 1024 + (r & 7) * 128;
        const int sw = r & 7;
        // This thread's bytes of stage `pset` in a packed-bit buffer.  I8: 32-byte rows, TMA 32-byte swizzle
        // (16-byte halves swapped on odd groups of 4 rows).  FP4: 64-byte rows, TMA 64-byte swizzle (16-byte
        // chunk index ^ (row/2 mod 4)); the thread reads chunks 2*pset and 2*pset+1.
        const uint32_t bits_row = smem0 + T::OFF_BITS + prow * T::BITS_ROW_BYTES;
        const uint32_t bits_c0 = KIND == KIND_FP4 ? (((2u * pset) ^ ((prow >> 1) & 3)) << 4)
                                                  : (((uint32_t)pset ^ ((prow >> 2) & 1)) << 4);
        const uint32_t bits_c1 = ((2u * pset + 1) ^ ((prow >> 1) & 3)) << 4;   // FP4 only
        const bool a_tmem = T::A_TMEM && isA;          // warp-uniform: warps 0-3 and 8-11 hold the A rows
        const uint32_t a_taddr0 = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + T::TMEM_A;
        const uint32_t full_leader0 = map_to_cta(full0, 0);
        const uint32_t tmem_empty_leader = map_to_cta(tmem_empty, 0);
        const int q4 = warp & 3;                      // TMEM lane quarter this warp may read
        const int cq = warp >> 2;                     // which 64 accumulator columns it drains
        uint32_t tphase = 0;                          // parity of tmem_full
        int epi_I = -1, epi_J = -1, epi_t = -1;       // tile whose accumulators still wait for their epilogue
        unsigned int chunks_seen = 0;                 // host-copy gate: chunks known to have landed

        // Publish this set's stage that is written but not yet visible to the MMA thread.
        auto publish_pending = [&]() {
            if (pending < 0) return;
            if (a_tmem) {
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                tc_fence_before();
            } else {
                fence_proxy_async_smem();
            }
            __syncwarp();
            if (lane == 0 && !(dbg & 64)) mbar_arrive_cluster(full_leader0 + 8 * pending);
            pending = -1;
        };
        // Fused epilogue of tile (eI, eJ) (eI still carries the set index of a batch): TMEM -> registers -> mask by
        // R[i][j], i<j -> histogram.
        auto epilogue = [&](int eIs, int eJ, int et) {
            if (dbg & 64) return;
            const int eI = eIs & TILE_I_MASK, eset = BATCH ? eIs >> TC_SET_SHIFT : 0;
            const long long i0 = (long long)eI * TC_T, j0 = (long long)eJ * TC_T;
            const long long i = i0 + 128 * (int)rank + 32 * q4 + lane;
            const uint32_t* relrow32 = reinterpret_cast<const uint32_t*>(rel + ((long long)eset * N + (i < N ? i : 0)) * stride_words);
            unsigned long long* const set_counts = counts + (long long)eset * (BATCH ? counts_stride : 0);   // batch: this set's abundances
            uint32_t relw[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {             // relation bits first: their latency hides behind the wait
                const long long jc = j0 + 32 * (2 * cq + e);
                uint32_t rw = (i < N) ? __ldg(relrow32 + (jc >> 5)) : 0u;
                if (jc + 31 <= i) rw = 0u;            // keep only columns j > i
                else if (jc <= i) rw &= 0xFFFFFFFFu << (int)(i - jc + 1);
                relw[e] = rw;
            }
            mbar_wait(tmem_full, tphase);
            tphase ^= 1;
            tc_fence_after();
            // Both 32-column chunks of this thread go to registers first; the accumulators are then handed back to the MMA
            // thread (tmem_empty) BEFORE the values are looked at, so the next tile's MMAs -- their first stages are already
            // in the ring -- run while this tile is bucketed.  The accumulator encodes n_ij monotonically (fp4: the f32 bit
            // pattern of 4 n, int8: n << 2TB), so "n <= kmax" is one unsigned compare against vmax with no conversion
            // (F2I runs at a quarter of the ALU rate and made the epilogue the longest part of a tile boundary); only the
            // values that pass are decoded.
            const int kcap = (int)min((long long)kmax, N - 2 < 0 ? 0LL : N - 2);       // n_ij never exceeds N-2
            const uint32_t vmax = KIND == KIND_FP4 ? __float_as_uint(4.0f * (float)kcap) : ((uint32_t)kcap << (2 * TB));
            uint32_t v0[32], v1[32];
            tmem_ld_32x32(tmem_base + ((uint32_t)(32 * q4) << 16) + (uint32_t)(32 * (2 * cq)), v0);
            tmem_ld_32x32(tmem_base + ((uint32_t)(32 * q4) << 16) + (uint32_t)(32 * (2 * cq + 1)), v1);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(tmem_empty_leader);
            // General bucketing (any kmax): one test per value.  Measured alternatives (config 3, ms per launch): this loop 89.65; a
            // branch-free pass that builds a 32-bit mask of passing values (compare + select + add) and then visits the
            // set bits eight at a time 91.80 -- per WARP nearly every group of columns holds a hit, so the second pass
            // branches as often; the same mask with the values copied to a local-memory scratch and a loop over the set
            // bits 94.3; no bucketing at all (wrong counts) 85.30.
            auto bucket = [&](uint32_t v) {
                // fp4: 4 n < 2^24 is an exact f32; n = low 23 bits of (4n * 0.25 + 2^23)
                const int n = KIND == KIND_FP4 ? (int)(__float_as_uint(fmaf(__uint_as_float(v), 0.25f, 8388608.0f)) & 0x7FFFFFu)
                                               : (int)(v >> (2 * TB));
                if (n < hist_bins && !BATCH) atomicAdd(&hist[n], 1u);
                else atomicAdd(&set_counts[n], 1ULL);
            };
            // Local action (kmax <= 3, every BASELINE.json config but the smeared one): no branch and no atomic per value.
            // Each thread keeps the four bins in the four bytes of one register (it sees 64 values per tile, so a byte
            // cannot overflow) and adds "1 << 8n" for every related pair; PTX shl clamps shift amounts above 31, so the
            // term is 0 for every n >= 4.  The pass is bound by the ALU pipe (16 lanes per scheduler, 4 warps each), so
            // what counts is ALU instructions per value -- 2.5 now, from 4:
            //   * 8n straight from the accumulator's bit pattern by ONE multiplication (FMA pipe): the f32 accumulator
            //     holds 4n, and 4n * 2^-148 = 8n * 2^-149 is a subnormal whose bit pattern IS the integer 8n (exact;
            //     for 8n >= 2^23 the product is a normal number with a pattern >= 2^23, which the shift clamps away like
            //     every other n >= 4).  Needs subnormals, i.e. no -ftz / fast-math (the build has neither).  Before:
            //     FFMA with 2^23 + AND with the mantissa mask;
            //   * the relation bit goes into bit 31 of the shift amount (x-th bit of ~rw moved up by an IMAD.SHL on the
            //     FMA pipe, merged by one LOP3), so an unrelated pair shifts the 1 out as well -- no mask, no predicate;
            //   * int8 kind: a shift of the s32 accumulator instead of the multiplication.
            // Measured on one box, config 1 / 2 / 3: 0.2525 / 10.85 / 81.67 ms -> 0.2382 / 10.66 / 80.83 ms; without any
            // bucketing (wrong counts) 0.200 / - / 78.3.  The four bytes are summed over the warp once per tile (4 REDUX +
            // at most 4 shared-memory atomics per warp).
            const bool byte_bins = !DUMP && kcap <= 3 && N <= (1LL << 20);
            if (byte_bins) {
                uint32_t packed = 0u;
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    if (dbg & 8) break;               // ablation: no bucketing (the accumulators are still read)
                    const uint32_t rw = relw[e];
                    if (rw == 0u) continue;           // no related pair among these 32 columns
#pragma unroll
                    for (int x = 0; x < 32; ++x) {
                        const uint32_t v = e == 0 ? v0[x] : v1[x];
                        const uint32_t sh = KIND == KIND_FP4 ? __float_as_uint(__fmul_rn(__uint_as_float(v), __uint_as_float(2u)))
                                                             : (v >> (2 * TB - 3));
                        const uint32_t amt = sh | ((~rw << (31 - x)) & 0x80000000u);   // bit 31: not a related pair
                        uint32_t onehot;
                        asm("shl.b32 %0, 1, %1;" : "=r"(onehot) : "r"(amt));     // 0 when 8 n > 31 or unrelated
                        packed += onehot;
                    }
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const unsigned int c = __reduce_add_sync(0xFFFFFFFFu, (packed >> (8 * k)) & 0xFFu);
                    if (lane == 0 && c != 0u && k <= kcap) {
                        if (!BATCH) atomicAdd(&hist[k], c);
                        else atomicAdd(&set_counts[k], (unsigned long long)c);
                    }
                }
            } else {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                if (dbg & 8) break;                   // ablation: no bucketing (the accumulators are still read)
                const uint32_t rw = relw[e];
                if (!DUMP && rw == 0u) continue;      // no related pair among these 32 columns
#pragma unroll
                for (int x = 0; x < 32; ++x) {
                    const uint32_t v = e == 0 ? v0[x] : v1[x];
                    if (DUMP) {                       // test hook: every n_ij of the tile, -1 where i, j are not a related pair
                        const int n = KIND == KIND_FP4 ? (int)(__uint_as_float(v) * 0.25f) : (int)(v >> (2 * TB));
                        dump[((size_t)et * TC_T + (size_t)(128 * (int)rank + 32 * q4 + lane)) * TC_T + 32 * (2 * cq + e) + x] =
                            ((rw >> x) & 1u) ? n : -1;
                    } else if ((rw & (1u << x)) && v <= vmax) {
                        bucket(v);
                    }
                }
            }
            }
            // one count per finished tile of this cluster (throttle of the TMA threads, see below)
            if (progress != nullptr && rank == 0 && tid == 0) atomicAdd(progress, 1u);
        };

        for (int rd = 0; rd < rounds; ++rd) {
            const int t = rd * G + ((rd & 1) ? (G - 1 - cl) : cl);
            if (t >= ntiles) continue;
            const int2 tile = tiles[t];
            const int I = tile.x & TILE_I_MASK, J = tile.y;
            int kb_begin, kb_end;                     // stages of COLS columns, [begin, end): even count
            tile_k_range<COLS>(I, J, kb_begin, kb_end);
            const int kbA = (256 * I + 255) / COLS;   // stages kb <= kbA can hold columns k <= i
            const int kbB = (256 * J) / COLS;         // stages kb >= kbB can hold columns k >= j

            // Software pipeline: the fence + arrive that publishes a stage is issued after the ALU work of this
            // set's next stage (its stores have drained by then); the empty-slot barrier is probed before that work.
            // Order of work: ... stages of tile t | first TC_PREFILL_GROUPS groups of tile t+1 | epilogue of tile t |
            // rest of tile t+1 ...  While the accumulators of tile t are drained (the MMA thread waits for tmem_empty)
            // the ring already holds the first stages of tile t+1, so the tensor cores restart at once and the
            // producers get those stages' time to refill their pipeline.
            const int prefill = (dbg & 128) ? 0 : TC_PREFILL_GROUPS;    // dbg 128: epilogue before any next stage
            if (prefill == 0 && epi_I >= 0) {
                publish_pending();
                epilogue(epi_I, epi_J, epi_t);
                epi_I = -1;
            }
            int gdone = 0;                            // live groups of this tile expanded so far
            if (GATE && SPARSE && landed != nullptr && occ != nullptr) wait_landed(landed, (unsigned int)tile_need[t], chunks_seen);
            // One stage of one row: open-range mask, expansion, publish of this warp's previous stage, store.
            auto do_stage = [&](int kb, uint32_t stage, uint32_t eparity, uint32_t (&w)[WORDS]) {
                if (dbg & 256) {                              // ablation: no open-range masks
                } else if (isA) {
                    if (kb <= kbA) {                          // keep k > i
                        const int rl = 256 * I + rt - COLS * kb;
#pragma unroll
                        for (int m = 0; m < WORDS; ++m) w[m] &= keep_gt(rl, m);
                    }
                } else if (kb >= kbB) {                       // keep k < j
                    const int lim = 256 * J + rt - COLS * kb;
#pragma unroll
                    for (int m = 0; m < WORDS; ++m) w[m] &= keep_lt(lim, m);
                }
                const bool slot_free = (dbg & 64) ? true : mbar_try(empty0 + 8 * stage, eparity);   // 64: free-running producers
                uint4 o[8];
                if (dbg & 2) {                                // ablation: no expansion arithmetic
#pragma unroll
                    for (int m = 0; m < 8; ++m) o[m] = make_uint4(w[m % WORDS], w[(m + 1) % WORDS], w[(m + 2) % WORDS], w[(m + 3) % WORDS]);
                } else if (KIND == KIND_FP4) {
                    unpack_group_fp4(&w[0], &o[0]);
                    unpack_group_fp4(&w[WORDS - 4], &o[4]);
                } else {
#pragma unroll
                    for (int m = 0; m < 4; ++m) unpack_word<TB>(w[m], o[2 * m], o[2 * m + 1]);
                }
                if (pending >= 0) {                           // publish this warp's previous stage to the leader's MMA thread
                    if (dbg & 16) {}                          // ablation: no fence before the publish
                    else if (a_tmem) tmem_wait_st_after(o);
                    else fence_proxy_async_smem_after(o);
                    __syncwarp();
                    if (lane == 0 && !(dbg & 64)) mbar_arrive_cluster(full_leader0 + 8 * pending);
                }
                if (!slot_free) mbar_wait(empty0 + 8 * stage, eparity);
                if (dbg & 4) {                                 // ablation: no operand stores
                } else if (a_tmem) {
                    tc_fence_after();                          // the MMAs that read this TMEM slot have completed
                    tmem_st_32x32(a_taddr0 + 32u * stage, o);
                } else {
                    const uint32_t rowp = row_smem + stage * T::STAGE_BYTES;
#pragma unroll
                    for (int c = 0; c < 8; ++c) sts128(rowp + ((c ^ sw) << 4), o[c]);
                }
                pending = (int)stage;
            };
            for_live_groups<SPARSE, GATE>(occ, occ_stride, I, J, kb_begin, kb_end, [&](int kb0) {
                // The packed-bit buffer is released only after the operand stores that consume every word loaded from
                // it: the hardware has then issued them after the LDS data arrived.  An arrive placed right after the
                // LDS instructions is NOT ordered after their completion (naming the loaded registers as unused asm
                // operands creates no dependency in the machine code), and with the ring full the TMA thread refills
                // the buffer at once: when the shared-memory pipe was backed up (the epilogue's histogram atomics of
                // slower warps) the delayed LDS returned the bits of the group four ahead.  Seen as a handful of wrong
                // n_ij per 10^10 pairs at config 4, and as thousands when the epilogue of a tile overlapped the first
                // stages of the next; located by dumping every n_ij and matching the wrong rows against "same row,
                // packed bits of the stage 8 later".
                if (TC_WHOLE_GROUP) {
                    // set p expands BOTH stages of every second group: one buffer wait, one release and one pass
                    // through the loop overhead per two stages
                    if ((int)(gsel & 1u) == pset) {
                        uint32_t w0[WORDS], w1[WORDS];
                        const bool ring = !(dbg & 32);
                        if (ring) {
                            mbar_wait(bits_full0 + 8 * bb, bphase);
                            const uint32_t base = bits_row + bb * T::BITS_BUF_BYTES;
                            if (KIND == KIND_FP4) {
                                const uint32_t z = (prow >> 1) & 3;
                                const uint4 v0 = lds128(base + ((0u ^ z) << 4)), v1 = lds128(base + ((1u ^ z) << 4));
                                const uint4 v2 = lds128(base + ((2u ^ z) << 4)), v3 = lds128(base + ((3u ^ z) << 4));
                                w0[0] = v0.x; w0[1] = v0.y; w0[2] = v0.z; w0[3] = v0.w;
                                w0[WORDS - 4] = v1.x; w0[WORDS - 3] = v1.y; w0[WORDS - 2] = v1.z; w0[WORDS - 1] = v1.w;
                                w1[0] = v2.x; w1[1] = v2.y; w1[2] = v2.z; w1[3] = v2.w;
                                w1[WORDS - 4] = v3.x; w1[WORDS - 3] = v3.y; w1[WORDS - 2] = v3.z; w1[WORDS - 1] = v3.w;
                            } else {
                                const uint32_t z = (prow >> 2) & 1;
                                const uint4 v0 = lds128(base + ((0u ^ z) << 4)), v1 = lds128(base + ((1u ^ z) << 4));
                                w0[0] = v0.x; w0[1] = v0.y; w0[2] = v0.z; w0[3] = v0.w;
                                w1[0] = v1.x; w1[1] = v1.y; w1[2] = v1.z; w1[3] = v1.w;
                            }
                        } else {
#pragma unroll
                            for (int m = 0; m < WORDS; ++m) { w0[m] = 0x01234567u * (m + kb0); w1[m] = 0x089abcdu * (m + kb0); }
                        }
                        do_stage(kb0, slot0, spar ^ 1, w0);
                        do_stage(kb0 + 1, slot0 + 1, spar ^ 1, w1);
                        __syncwarp();
                        if (ring && lane == 0) mbar_arrive(bits_empty0 + 8 * bb);
                    }
                    ++gsel;
                    slot0 += 2;
                    if (slot0 == (uint32_t)T::STAGES) { slot0 = 0; spar ^= 1; }
                    if (++bb == T::BITS_BUFS) { bb = 0; bphase ^= 1; }
                } else {
                    const uint32_t stage = pset + 2 * sl;
                    const int kb = kb0 + pset;
                    uint32_t w[WORDS];
                    uint32_t bits_release = 0;
                    if (dbg & 32) {                               // ablation: no packed-bit ring
#pragma unroll
                        for (int m = 0; m < WORDS; ++m) w[m] = 0x01234567u * (m + kb);
                    } else {
                        mbar_wait(bits_full0 + 8 * bb, bphase);
                        const uint4 v0 = lds128(bits_row + bb * T::BITS_BUF_BYTES + bits_c0);
                        w[0] = v0.x; w[1] = v0.y; w[2] = v0.z; w[3] = v0.w;
                        if (KIND == KIND_FP4) {
                            const uint4 v1 = lds128(bits_row + bb * T::BITS_BUF_BYTES + bits_c1);
                            w[WORDS - 4] = v1.x; w[WORDS - 3] = v1.y; w[WORDS - 2] = v1.z; w[WORDS - 1] = v1.w;
                        }
                        bits_release = bits_empty0 + 8 * bb;
                        if (++bb == T::BITS_BUFS) { bb = 0; bphase ^= 1; }
                    }
                    do_stage(kb, stage, sphase ^ 1, w);
                    if (++sl == T::STAGES / 2) { sl = 0; sphase ^= 1; }
                    __syncwarp();
                    if (bits_release != 0 && lane == 0) mbar_arrive(bits_release);
                }
                if (epi_I >= 0 && ++gdone == prefill) {        // the previous tile's epilogue, after the prefill
                    publish_pending();
                    epilogue(epi_I, epi_J, epi_t);
                    epi_I = -1;
                }
            });
            if (epi_I >= 0) {                                  // this tile had fewer live groups than the prefill
                publish_pending();
                epilogue(epi_I, epi_J, epi_t);
            }
            epi_I = tile.x;                                    // with the set index of a batch
            epi_J = J;
            epi_t = t;
        }
        publish_pending();                                     // last stage of the last tile
        if (epi_I >= 0) epilogue(epi_I, epi_J, epi_t);
    } else if (warp == TC_MMA_WARP) {
        // ================================================================== MMA issuer (leader CTA, one elected lane issues)
        // The whole warp walks the loop converged (the barrier waits and the ring bookkeeping are warp-uniform, so they
        // stay on the uniform datapath); only the tcgen05 instructions sit under the elected lane's predicate.  This
        // one warp paces the tensor cores of two SMs: at ~88 instructions per stage (lane-0 branch, per-instruction
        // ELECT loops, descriptors rebuilt and moved to uniform registers every stage) it needed ~700 clk per stage
        // and was the bottleneck of the kernel (ncu source view: the warp never waited on `full`, it was busy issuing).
        if (rank == 0 && !(dbg & 64)) {
            const bool issuer = elect_one();
            uint32_t stage = 0, sphase = 0, ephase = 0;
            int done_tiles = 0;
            unsigned int chunks_seen = 0;
            const uint32_t tmem_sfa = tmem_base + T::TMEM_SF, tmem_sfb = tmem_base + T::TMEM_SFB;
            const uint64_t adesc0 = make_kmajor_sw128_desc(smem0), bdesc0 = make_kmajor_sw128_desc(smem0 + T::OFF_B);
            for (int rd = 0; rd < rounds; ++rd) {
                const int t = rd * G + ((rd & 1) ? (G - 1 - cl) : cl);
                if (t >= ntiles) continue;
                const int2 tile = tiles[t];
                int kb_begin, kb_end;
                const int tI = tile.x & TILE_I_MASK;
                tile_k_range<COLS>(tI, tile.y, kb_begin, kb_end);
                if (done_tiles > 0) {                       // both CTAs' accumulators must have been drained
                    mbar_wait(tmem_empty, ephase);
                    ephase ^= 1;
                }
                tc_fence_after();
                uint32_t fresh = 1;                         // the tile's first MMA overwrites the accumulators
                if (GATE && SPARSE && landed != nullptr && occ != nullptr) wait_landed(landed, (unsigned int)tile_need[t], chunks_seen);
                for_live_groups<SPARSE, GATE>(occ, occ_stride, tI, tile.y, kb_begin, kb_end, [&](int) {
#pragma unroll 1
                for (int st = 0; st < TC_GROUP; ++st) {
                    mbar_wait(full0 + 8 * stage, sphase);
                    tc_fence_after();
                    if (issuer) {
                        const uint64_t soff = (uint64_t)(stage * (T::STAGE_BYTES >> 4));   // descriptor address unit: 16 bytes
                        const uint64_t adesc = adesc0 + soff, bdesc = bdesc0 + soff;
                        const uint32_t a_tmem = tmem_base + T::TMEM_A + 32u * stage;
#pragma unroll
                        for (int kk = 0; kk < TC_ROW_BYTES / 32; ++kk) {   // 32 bytes of K per instruction: +2 in 16-byte units
                            const uint32_t acc = kk > 0 ? 1u : (fresh ^ 1u);
                            if (dbg & 1) continue;                          // ablation: no MMA issue
                            const uint32_t idesc4 = (kk & 1) ? TC_IDESC_FP4_ODD : TC_IDESC_FP4;   // which two scale bytes
                            if (KIND == KIND_FP4 && T::A_TMEM)
                                umma_mxf4_2cta_ts(tmem_base, a_tmem + 8u * kk, bdesc + 2 * kk, idesc4, acc, tmem_sfa, tmem_sfb);
                            else if (KIND == KIND_FP4)
                                umma_mxf4_2cta(tmem_base, adesc + 2 * kk, bdesc + 2 * kk, idesc4, acc, tmem_sfa, tmem_sfb);
                            else
                                umma_i8_2cta(tmem_base, adesc + 2 * kk, bdesc + 2 * kk, TC_IDESC, acc);
                        }
                        umma_commit_2cta(empty0 + 8 * stage);
                    }
                    fresh = 0;
                    if (++stage == T::STAGES) { stage = 0; sphase ^= 1; }
                }
                });
                if (issuer) umma_commit_2cta(tmem_full);     // arrives when every MMA of the tile has completed
                ++done_tiles;
            }
        }
    } else {
        // ================================================================== TMA warp: packed bits -> shared ring
        if (lane == 0) {
            uint32_t bb = 0, bphase = 0;
            bool throttling = true;
            unsigned int chunks_seen = 0;
            for (int rd = 0; rd < rounds; ++rd) {
                const int t = rd * G + ((rd & 1) ? (G - 1 - cl) : cl);
                if (t >= ntiles) continue;
                const int2 tile = tiles[t];
                const int tI = tile.x & TILE_I_MASK;
                const int set_row0 = BATCH ? (tile.x >> TC_SET_SHIFT) * (int)N : 0;   // first row of the tile's causal set
                const int ia = set_row0 + tI * TC_T + 128 * (int)rank, jb = set_row0 + tile.y * TC_T + 128 * (int)rank;
                int kb_begin, kb_end;
                tile_k_range<COLS>(tI, tile.y, kb_begin, kb_end);
                // Keep the clusters within TC_MAX_LEAD rounds of the average: the schedule has no barrier between rounds,
                // and with a slow, variable epilogue (full histogram) the clusters of a patch drift apart until none of
                // them shares row segments in L2 any more (config 4: 2.55 TB of DRAM reads per launch, L2 hit rate
                // 38 %).  A cluster starts round rd only when (rd - TC_MAX_LEAD) * G tiles are finished in total; the
                // slowest cluster never waits (everybody else has finished at least as many), so no deadlock, and the
                // makespan of the static deal is unchanged.  Only the TMA thread polls; everything downstream starves.
                // The wait is bounded: it relies on all clusters of the grid being resident together (the host clamps the
                // grid to cudaOccupancyMaxActiveClusters), and if that ever fails -- SMs held by another kernel or an MPS
                // limit -- a cluster that has polled TC_THROTTLE_MAX_POLLS times in one wait (> 6.5 ms; a tile takes well
                // under 1 ms) stops throttling for the rest of the launch: the failure costs L2 reuse, not a hang.
                if (WAITS && progress != nullptr && rd > TC_MAX_LEAD && throttling) {
                    const unsigned int need = (unsigned int)(rd - TC_MAX_LEAD) * (unsigned int)G;
                    int polls = 0;
                    while (*reinterpret_cast<volatile unsigned int*>(progress) < need) {
                        if (++polls >= TC_THROTTLE_MAX_POLLS) { throttling = false; break; }
                        __nanosleep(200);
                    }
                }
                // Host-copy gate (wait_landed above).
                if (GATE && landed != nullptr) {
                    const unsigned int before = chunks_seen;
                    wait_landed(landed, (unsigned int)tile_need[t], chunks_seen);
                    if (chunks_seen != before) asm volatile("fence.proxy.async.global;" ::: "memory");   // the bytes are read by the async proxy (TMA)
                }
                if (!(dbg & 32)) for_live_groups<SPARSE, GATE>(occ, occ_stride, tI, tile.y, kb_begin, kb_end, [&](int kb0) {
                    mbar_wait(bits_empty0 + 8 * bb, bphase ^ 1);
                    const uint32_t bar = bits_full0 + 8 * bb;
                    const uint32_t dst = smem0 + T::OFF_BITS + bb * T::BITS_BUF_BYTES;
                    mbar_expect_tx(bar, T::BITS_BUF_BYTES);
                    tma_load_2d(dst, &bits_map, kb0 * (COLS / 8), ia, bar);
                    tma_load_2d(dst + T::BITS_BOX_BYTES, &bits_map, kb0 * (COLS / 8), jb, bar);
                    if (++bb == T::BITS_BUFS) { bb = 0; bphase ^= 1; }
                });
            }
        }
    }

    // ---- teardown: flush the privatised histogram, release TMEM once neither CTA can touch the other any more
    tc_fence_before();
    __syncthreads();
    for (int b = tid; b < hist_bins && b <= kmax; b += TC_THREADS)
        if (hist[b]) atomicAdd(&counts[b], (unsigned long long)hist[b]);
    cluster_sync_all();
    tc_fence_after();
    if (warp == TC_MMA_WARP) {
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(T::TMEM_COLS)
                     : "memory");
    }
}

}  // namespace csg
