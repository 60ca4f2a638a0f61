/*
 * csg.h -- C ABI of libcsg: Benincasa-Dowker action of a causal set on one B200 (sm_100a).
 *
 * The library computes the O(N^3) hot path of Cunningham & Krioukov, "Causal Set Generator and Action
 * Computer" (arXiv:1709.03013; citations below are /root/reference/PAPER.md:<line>):
 *   for every related pair i<j of a time-sorted causal set, the number n_ij of elements k with
 *   i < k < j related to both (Sec. 4.1; Fig. 2 caption; Algorithm 5,
 *   PAPER.md:407), the histogram N_k of those interval sizes, and the action built from it
 *   (Eq. 4; Eq. 5).
 *
 * Relation-matrix layout (FastBitset rows): N rows of csg_row_stride_words(N) 64-bit
 * words; bit c of row r is bit (c % 64), LSB first, of word r*stride + c/64.  The matrix
 * is symmetric (bit (r,c) == bit (c,r) == 1 iff the two elements are related), has a zero diagonal and zero
 * padding bits, and rows are sorted so that "r precedes c" implies r < c.  For a pair i<j the
 * library reads bit (i,j), bits (i,k) and bits (j,k) for i<k<j -- both triangles are used.
 *
 * No function throws; every function returns a CSG_* code (0 = success) unless stated otherwise.
 * There is no CPU fallback: without a CUDA device every compute entry point returns CSG_E_CUDA.
 * Pointers are tagged DEVICE or HOST.  The caller owns every buffer it passes; the library keeps a small
 * cached device workspace (tile schedules, counters, events) that csg_shutdown() frees.  Inputs are never modified.
 *
 * Devices and threads.  Every call works on the CURRENT CUDA device (cudaGetDevice); DEVICE pointers and the stream
 * must belong to it.  Cached state is kept per device, so one process may drive several GPUs (switch devices with
 * cudaSetDevice between calls).  The entry points are thread-safe (one internal mutex; they only enqueue work).
 * Stream-ordered calls (csg_action, csg_action_partial/_finish, csg_action_batch, csg_link, csg_interval_sizes) may
 * be in flight on different streams at the same time: cached tile schedules are immutable once built and are never
 * freed or rebuilt before csg_shutdown().  The HOST-buffer calls (csg_action_host, csg_causet_action_host) run on
 * an internal stream per device, share library-owned device buffers and return synchronised; they serialise.
 * csg_shutdown() must not be called while work of this library is still in flight, and it invalidates every CUDA
 * graph that captured a call of this library (the graph holds pointers into the cached workspace).
 * Per-launch scratch (the finished-tile counter of the drift throttle, the occupancy map of the block-sparse sweep)
 * comes from rings of 32 slots per device: at most 32 launches that use them may be in flight at once, and a graph
 * that captured such a launch (matrices of 96 MiB and more) keeps its slot, so it must not be replayed while 32 or more
 * later launches of the same kind are still running.
 */
#ifndef CSG_H_
#define CSG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#ifndef __DRIVER_TYPES_H__
typedef struct CUstream_st *cudaStream_t;
#endif

enum {
    CSG_OK = 0,
    CSG_E_NULL = -1,        /* a required pointer is NULL */
    CSG_E_SIZE = -2,        /* N < 1, N > CSG_MAX_N, npairs < 0, a tile index outside the matrix, iters < 1 */
    CSG_E_ALIGN = -3,       /* rel_bits not 16-byte aligned, counts/S not 8-byte aligned */
    CSG_E_DIM = -4,         /* dim not in {2, 4} */
    CSG_E_EPS = -5,         /* eps NaN or outside (0, 1] */
    CSG_E_KMAX = -6,        /* kmax < 0, kmax > CSG_MAX_KMAX, or too small for the local action */
    CSG_E_UNSUPPORTED = -7, /* csg_tile_interval_sizes while the bitset variant is selected */
    CSG_E_CUDA = -8,        /* a CUDA call failed; csg_strerror(CSG_E_CUDA) carries its text */
    CSG_E_VARIANT = -9,     /* unknown variant id or mode */
    CSG_E_SHARD = -10,      /* nshards < 1 or shard outside [0, nshards) */
    CSG_E_GEOMETRY = -11,   /* unknown geometry id */
    CSG_E_NOALLOC_LIMIT = -12 /* csg_action_noalloc: N > CSG_NOALLOC_MAX_N or kmax > CSG_NOALLOC_MAX_KMAX */
};

#define CSG_MAX_N (1 << 22)
#define CSG_MAX_KMAX (1 << 22)
#define CSG_MAX_BATCH 65535

enum {
    CSG_VARIANT_AUTO = 0,   /* fp4 tensor variant when N > 1024, else bitset (csg_action_batch: N > 128) */
    CSG_VARIANT_BITSET = 1, /* LOP3 AND + POPC over packed 32-bit words, register micro-tiles */
    CSG_VARIANT_TENSOR = 2, /* bits unpacked to u8 in shared memory, tcgen05.mma kind::i8, s32 accumulators in TMEM */
    CSG_VARIANT_TENSOR_FP4 = 3 /* bits unpacked to e2m1 nibbles, tcgen05.mma kind::mxf4 with unit block scales, f32
                                  accumulators (exact: every partial sum is an integer below 2^24) */
};

/* Row stride of the relation matrix in 64-bit words: 4*ceil(N/256) (rows 256-bit aligned). */
int64_t csg_row_stride_words(int64_t N);

/*
 * Interval abundances and action of one causal set.  All work is enqueued on `stream`.  The FIRST call for a new
 * (device, N) builds that size's tile schedule and copies it to the device with one blocking cudaMemcpy; every later
 * call with that N -- whatever other sizes were run in between, on whatever stream -- only enqueues a memset and
 * two or three kernels (small sets: one), synchronises nothing, and can be captured in a CUDA graph.
 *
 *   rel_bits DEVICE, N*csg_row_stride_words(N) words, layout above, 16-byte aligned, read only.
 *   N        number of elements, 1 <= N <= CSG_MAX_N (N = 1, 2 are valid: no triples).
 *   dim      2 or 4: which combination of abundances gives S.
 *   eps      1.0 -> local action: dim 2: S = 2(N - 2N_0 + 4N_1 - 2N_2) (Eq. 4 with n_i = N_{i-1});
 *                   dim 4: S = (4/sqrt 6)(N - N_0 + 9N_1 - 16N_2 + 8N_3) (not in the paper; A8).
 *                   Needs kmax >= 2 (dim 2) or >= 3 (dim 4).
 *            0 < eps < 1 -> smeared action; pass kmax = N-2 for the full sum.
 *                   dim 2 (Eq. 5): S = 2 eps [N - 2 eps sum_{k=0..kmax} N_k f_2(k, eps)];
 *                   dim 4 (not in the paper; A9): S = (4/sqrt 6) sqrt(eps) [N - eps sum_k N_k f_4(k, eps)],
 *                   f_4(k,e) = (1-e)^k [1 - 9ek/(1-e) + 8e^2 k(k-1)/(1-e)^2 - (4/3) e^3 k(k-1)(k-2)/(1-e)^3].
 *   kmax     highest interval size that is histogrammed; related pairs with n_ij > kmax are not counted.
 *   counts   DEVICE, kmax+1 int64, overwritten: counts[k] = N_k = number of related pairs i<j with exactly
 *            k elements strictly between (0-based; the paper's n_i is counts[i-1]).
 *   S        DEVICE, 1 double, overwritten.
 */
int csg_action(const uint64_t *rel_bits, int64_t N, int dim, double eps, int kmax, int64_t *counts,
               double *S, cudaStream_t stream);

/*
 * csg_action for callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc.  Same arguments, same results (counts bit-identical, S identical) as csg_action, for small causal
 * sets only:  N <= CSG_NOALLOC_MAX_N and kmax <= CSG_NOALLOC_MAX_KMAX, else CSG_E_NOALLOC_LIMIT (nothing is enqueued).
 * It runs the fused small-set launch of the bitset variant (AND + POPC tiles, histogram and action in ONE kernel,
 * whatever csg_set_variant says) with that launch's workspace -- 1024 accumulator bins and the last-CTA ticket -- in a
 * file-scope `static __device__` array of 8448 bytes instead of a cudaMalloc'ed buffer; every GPU that loads
 * libcsg.so holds those bytes until the process exits.  The call enqueues one memset of that array (it keeps the last
 * call's contents) and one kernel on `stream`, synchronises nothing, and calls no cudaMalloc, cudaFree or allocating
 * library routine, on its first use either.
 * ALL calls on a device share the one array: calls that overlap on the GPU (two streams, two host threads' launches
 * in flight together, a captured graph replayed next to an eager call) race on it and return garbage.  Keep them on one
 * stream or otherwise ordered.
 * csg_noalloc_setup(): optional; resolves the array's device address (cudaGetSymbolAddress) and reads the SM count for
 * the CURRENT device, once per device.  csg_action_noalloc does the same on its first call per device; call the
 * set-up yourself, with the device current, before a capture or a loop that must not touch the CUDA module loader.
 */
#define CSG_NOALLOC_MAX_N 4096
#define CSG_NOALLOC_MAX_KMAX 1023
int csg_noalloc_setup(void);
int csg_action_noalloc(const uint64_t *rel_bits, int64_t N, int dim, double eps, int kmax, int64_t *counts,
                       double *S, cudaStream_t stream);

/*
 * The same path in two halves, for one causal set whose pair tiles are split over several GPUs (the paper
 * splits the pair loop evenly over computers when the matrix fits on each, and reduces the
 * private histograms at the end).  Every GPU holds the whole relation matrix.
 *
 * csg_action_partial: steps a1-a3 over the tiles of shard `shard` of `nshards` (csg_tile_schedule):
 *   counts DEVICE, kmax+1 int64, overwritten with this shard's abundances.  The abundances of all shards
 *   add up to those of csg_action (the caller sums them, e.g. ncclAllReduce).  0 <= shard < nshards.
 * csg_action_finish: steps a4/a5 on summed abundances: counts DEVICE (read only), S DEVICE, 1 double;
 *   N, dim, eps, kmax as in csg_action.  csg_action == partial(shard 0 of 1) followed by finish.
 * Both enqueue on `stream` and do not synchronise (first call per (N, shard, nshards): as csg_action).
 * Which pairs a shard covers: tensor variants -- the tiles csg_tile_schedule lists for it; bitset variant (N <= 1024
 * under CSG_VARIANT_AUTO) -- every nshards-th 64 x 64 tile of its own depth-sorted enumeration, which
 * csg_tile_schedule does not describe.  Either way the shards of one N partition the related pairs exactly.
 */
int csg_action_partial(const uint64_t *rel_bits, int64_t N, int kmax, int shard, int nshards, int64_t *counts,
                       cudaStream_t stream);
int csg_action_finish(const int64_t *counts, int64_t N, int dim, double eps, int kmax, double *S,
                      cudaStream_t stream);

/*
 * A batch of causal sets of the same size in one call (Monte-Carlo chains and ensemble averages work on many
 * sets of modest size: PAPER.md:35, 457, 490).  rel_bits DEVICE: `batch` matrices back to back, each
 * N*csg_row_stride_words(N) words; counts DEVICE: batch x (kmax+1) int64, row b = abundances of set b; S DEVICE:
 * batch doubles.  Other arguments as csg_action.  1 <= batch <= CSG_MAX_BATCH, batch * N < 2^31.  Under
 * CSG_VARIANT_AUTO: N <= 128: one launch of the bitset kernel (grid.y = set); above that persistent tensor-core
 * launches that each work through the tiles of a power-of-two number of sets, deepest first across those sets (64
 * sets: one launch; 100 sets: 64 + 32 + 4; no launch and no tail per set, and one cached tile list per power of two).
 * Only sets whose matrix exceeds 48 MiB run back to back, one launch each (they fill the machine on their own and
 * take the patch schedule and the block-sparse sweep).
 */
int csg_action_batch(const uint64_t *rel_bits, int64_t N, int64_t batch, int dim, double eps, int kmax,
                     int64_t *counts, double *S, cudaStream_t stream);

/*
 * Host logic, no device needed: the pair tiles (I, J), I <= J, in 256-row blocks, that shard `shard` of
 * `nshards` visits, in launch order (deepest K-range first; for matrices larger than L2 grouped in patches of
 * 8 x 9 blocks so that concurrently running tiles share rows in L2).  tiles_ij HOST, 2*capacity int32
 * (I0, J0, I1, J1, ...), may be NULL; returns the number of tiles of the shard (or a negative CSG_E_* code);
 * at most `capacity` tiles are written.  The shards of one N partition the upper triangle exactly.
 * Describes the tensor variants only (see csg_action_partial).
 */
int64_t csg_tile_schedule(int64_t N, int shard, int nshards, int32_t *tiles_ij, int64_t capacity);

/*
 * Same computation with HOST buffers (the end-to-end call): copies rel_bits to the device (pinned or
 * pageable host memory), runs csg_action on an internal stream, copies counts and S back and
 * synchronises.  rel_bits_host: N*stride words; counts_host: kmax+1 int64; S_host: 1 double.
 * Matrices of 32 MiB and more go over in 64 row chunks, outermost chunks first, on a copy stream while ONE
 * persistent launch of the interval kernel already runs: after each chunk the copy stream publishes how many have
 * been delivered (cuStreamWriteValue32) and a tile starts when the two row blocks it reads are there
 * (overlap of the transfer with the computation).  With the block-sparse sweep (csg_set_sparse) the
 * blocks of a chunk are marked by a small kernel on a third stream before the chunk is published, and the persistent
 * launch leaves one SM pair free for those kernels.
 */
int csg_action_host(const uint64_t *rel_bits_host, int64_t N, int dim, double eps, int kmax,
                    int64_t *counts_host, double *S_host);

/*
 * How csg_action_host overlaps the copy of a large matrix with the kernel.  CSG_HOST_PIPELINE_AUTO: the gated single
 * launch described above when the driver offers stream memory operations (fp4 kind), else chunked launches;
 * _CHUNKED: always one launch per copy step behind an event.  The gated launch WAITS inside the kernel for the copy
 * stream, so it needs copies and kernels to run concurrently: under a tool that serialises the GPU's work (Nsight
 * Compute replays one kernel at a time and holds every other stream) it cannot make progress -- select _CHUNKED for
 * such runs (bench.py --host-pipeline chunked).  The same holds for anything else that synchronises the whole context
 * while csg_action_host is running: CUDA loads kernels lazily, and the first launch of a not-yet-loaded kernel from
 * ANOTHER host thread may have to wait for the gated kernel, which waits for copies this call is still enqueueing.
 * (The library force-loads its own kernels before it launches a gated kernel.)  A process in which other threads may
 * launch new kernels during csg_action_host should select _CHUNKED or run with CUDA_MODULE_LOADING=EAGER.
 * Results never depend on the mode.
 */
enum { CSG_HOST_PIPELINE_AUTO = 0, CSG_HOST_PIPELINE_CHUNKED = 1 };
int csg_set_host_pipeline(int mode);

/*
 * Linking (Sec. 2.2: "pairwise relations are found by identifying pairs of elements which are
 * timelike separated"; dense, symmetric, topologically sorted adjacency matrix): builds the relation matrix
 * that csg_action reads from the coordinates of the elements.
 *
 *   coords   DEVICE, N rows of dim doubles, one row per element, ALREADY sorted by the time coordinate
 *            (first column), 8-byte aligned, read only.
 *   geometry CSG_GEOM_MINKOWSKI_2D: (u, v) light-cone coordinates; i<j related iff u_i<u_j and v_i<v_j.
 *            CSG_GEOM_MINKOWSKI_4D: (t, x, y, z); related iff dt>0 and dt*dt > (dx*dx+dy*dy)+dz*dz.
 *            CSG_GEOM_DESITTER_2D:  (eta, theta); related iff pi-|pi-|dtheta|| < |deta|.
 *            All in double, one rounding per operation, strict inequalities; the direction of a relation is
 *            the index order.  (The two Minkowski tests are not in the paper: DESIGN.md reading A17.)
 *   rel_bits DEVICE, N*csg_row_stride_words(N) words, 16-byte aligned; every word is overwritten (symmetric
 *            matrix, zero diagonal, zero padding).
 * Enqueued on `stream`, no host synchronisation.
 */
enum { CSG_GEOM_MINKOWSKI_2D = 0, CSG_GEOM_MINKOWSKI_4D = 1, CSG_GEOM_DESITTER_2D = 2 };
int csg_link(const double *coords, int64_t N, int geometry, uint64_t *rel_bits, cudaStream_t stream);

/*
 * Coordinates in, action out, with HOST buffers: copies the N x dim coordinates to the device (4 MiB at
 * N = 131072 in 4D instead of the 2 GiB matrix), csg_link into a library-owned matrix, csg_action (dim 2 for
 * the two (1+1) geometries, 4 for Minkowski 4D), copies counts and S back and synchronises.
 * coords_host: N*dim doubles, time-sorted; counts_host: kmax+1 int64; S_host: 1 double.
 */
int csg_causet_action_host(const double *coords_host, int64_t N, int geometry, double eps, int kmax,
                           int64_t *counts_host, double *S_host);
/* Milliseconds of the latest csg_link kernel launched while kernel timing was enabled (HOST float). */
int csg_last_link_ms(float *ms);

/*
 * Test hook: interval sizes of listed pairs.  pairs_ij DEVICE, 2*npairs int64 (i0, j0, i1, j1, ...);
 * n_out DEVICE, npairs int32: n_ij if 0 <= i < j < N and bit (i,j) is set, else -1.
 */
int csg_interval_sizes(const uint64_t *rel_bits, int64_t N, const int64_t *pairs_ij, int64_t npairs,
                       int32_t *n_out, cudaStream_t stream);

/*
 * Test hook for the tensor variants: every interval size of whole 256 x 256 tiles, computed by the SAME kernel,
 * tile sweep, open-range masks and accumulators as csg_action (its epilogue writes n_ij instead of bucketing it).
 * tiles_ij_host HOST, 2*ntiles int32 (I0, J0, I1, J1, ...), 256-row blocks with 0 <= I <= J < ceil(N/256);
 * n_out DEVICE, ntiles*256*256 int32: n_out[(t*256 + r)*256 + c] = n_ij for i = 256 I_t + r, j = 256 J_t + c if
 * i < j < N and bit (i,j) is set, else -1.  Uses the variant csg_action would use for this N (CSG_E_UNSUPPORTED
 * for the bitset variant).  Synchronises `stream` before it returns.  0 <= ntiles <= 32768.
 */
int csg_tile_interval_sizes(const uint64_t *rel_bits, int64_t N, const int32_t *tiles_ij_host, int64_t ntiles,
                            int32_t *n_out, cudaStream_t stream);

/* Choose the kernel variant for later csg_action calls (CSG_VARIANT_*); returns CSG_E_VARIANT if unknown. */
int csg_set_variant(int variant);
/* The variant csg_action would run for this N under the current setting (CSG_VARIANT_BITSET, _TENSOR or _TENSOR_FP4). */
int csg_effective_variant(int64_t N);

/*
 * Measurement / test aid like csg_set_variant: the drift throttle of the fp4 tensor kernel (clusters of the
 * persistent grid are kept within one round of each other so that concurrently running tiles share rows in L2).
 * CSG_THROTTLE_AUTO: on for matrices above 1 GiB only; _ON: on whenever a launch has more tiles than clusters;
 * _OFF: never.  In every mode it is used only if the runtime reports that the whole grid can be resident at once,
 * and a wait that lasts longer than a few ms switches it off inside the kernel.  Results never depend on it.
 */
enum { CSG_THROTTLE_AUTO = 0, CSG_THROTTLE_ON = 1, CSG_THROTTLE_OFF = 2 };
int csg_set_throttle(int mode);

/*
 * Block-sparse K sweep of the fp4 tensor kernel.  The paper's pair loop skips unrelated pairs (Algorithm 5
 * l.4-5), so its run time depends on the ordering fraction.  A tensor-core tile cannot skip single
 * pairs, but the stage of tile (I, J) that sweeps column block K multiplies the 256 x 256 block (I, K) of the matrix
 * with block (J, K) and contributes nothing when either is empty -- and in a time-sorted 3+1 sprinkling the blocks
 * next to the diagonal are (elements close in time are almost never timelike separated).  One pass over the matrix
 * marks the empty blocks (csg_block_occupancy) and the kernel neither fetches, expands nor multiplies the two-stage
 * groups (2 x 256 columns) in which both stages are dead; results never depend on it.
 * CSG_SPARSE_AUTO: matrices of 96 MiB and more (N >= 28000; below, the extra launch costs more than the dead
 * groups), unless the call says dim = 2 (a 1+1 order, flat or de Sitter, has
 * no empty block, and the pass and the mask loop would cost 2 %; csg_action_partial has no dim and uses the sweep);
 * _ON: every fp4 launch (test aid); _OFF: never.  csg_action_host marks the blocks of every chunk as it lands.
 */
enum { CSG_SPARSE_AUTO = 0, CSG_SPARSE_ON = 1, CSG_SPARSE_OFF = 2 };
int csg_set_sparse(int mode);
/*
 * The occupancy pass on its own (test hook and measurement aid).  occ DEVICE, ceil(N/256) rows of
 * csg_occupancy_stride_words(N) 32-bit words, every word overwritten: bit (K % 32) of word K / 32 of row I is set iff
 * some bit of rows 256 I .. 256 I + 255, columns 256 K .. 256 K + 255 of the matrix is set; words beyond the last
 * column block are zero.  rel_bits as in csg_action.  Enqueued on `stream`, no host synchronisation.
 */
int64_t csg_occupancy_stride_words(int64_t N);
int csg_block_occupancy(const uint64_t *rel_bits, int64_t N, uint32_t *occ, cudaStream_t stream);

/*
 * Measurement aid: the roofline denominators measured on the current device.  Runs a bare kernel (no producers, no
 * memory traffic) and returns its CUDA-event time in *ms (HOST) and the work it did in *units (HOST):
 *   CSG_PEAK_MMA_MXF4  the interval kernel's own instruction, tcgen05.mma.cta_group::2.kind::mxf4 block32, M = N = 256,
 *                      K = 64, A from TMEM, issued back to back by one thread per SM pair; units = MACs
 *   CSG_PEAK_MMA_I8    the same for kind::i8 (K = 32, both operands in shared memory); units = MACs
 *   CSG_PEAK_ALU_MIX   the bitset variant's inner mix, 1 AND + 1 POPC + 1 ADD per step on 32-bit words; units = lane-steps
 *                      (one lane-step = 32 ordered-triple tests)
 *   CSG_PEAK_ALU_POPC / CSG_PEAK_ALU_LOP3   one POPC / one LOP3 per step; units = lane-steps
 * iters: 4-MMA groups per SM pair (tensor) or loop trips of 8 steps per thread (ALU).  Synchronises the device.
 */
enum { CSG_PEAK_MMA_MXF4 = 0, CSG_PEAK_MMA_I8 = 1, CSG_PEAK_ALU_MIX = 2, CSG_PEAK_ALU_POPC = 3, CSG_PEAK_ALU_LOP3 = 4 };
int csg_measure_peak(int what, int iters, float *ms, double *units);

/*
 * Measurement aids.  csg_set_kernel_timing(1) makes csg_action bracket its dominant kernel (the interval
 * kernel, not the memsets or the finishing kernel) with CUDA events on the caller's stream;
 * csg_last_kernel_ms waits for those events and returns the elapsed milliseconds of the latest call.
 * csg_launch_count returns how many kernels this library has launched in this process.
 */
int csg_set_kernel_timing(int enable);
int csg_last_kernel_ms(float *ms);
/* Same for the latest n timed calls (1 <= n <= 64), oldest first: ms HOST, n floats.  CSG_E_CUDA if fewer
 * than n calls were timed since timing was enabled. */
int csg_kernel_ms_history(float *ms, int n);
int64_t csg_launch_count(void);

/* Text for a code; for CSG_E_CUDA it includes the text of the last CUDA error the library saw. */
const char *csg_strerror(int code);

/* Free the cached device workspace and internal stream/events.  Safe to call more than once. */
int csg_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* CSG_H_ */
