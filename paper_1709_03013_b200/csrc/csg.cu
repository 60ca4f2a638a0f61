// libcsg: C-ABI entry points (include/csg.h), argument validation, cached device workspace, tile
// schedule, finishing kernel.  Every step of the hot path runs in the kernels of this directory; there is
// no CPU fallback.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <map>
#include <mutex>
#include <vector>

#include "../../include/csg.h"
#include "finish.cuh"
#include "bitset_kernel.cuh"
#include "link_kernel.cuh"
#include "occupancy_kernel.cuh"
#include "tensor_kernel.cuh"
#include "peak_kernels.cuh"

namespace csg {

// ---------------------------------------------------------------------------------------------- finishing
// counts -> S (csrc/finish.cuh).  One CTA per causal set of a batch.
constexpr int FIN_THREADS = 1024;

__global__ void __launch_bounds__(FIN_THREADS, 1)
finish_action_kernel(const long long* __restrict__ counts, long long N, int dim, double eps, int kmax,
                     double* __restrict__ S) {
    __shared__ double red[FIN_LANES];
    finish_block(counts + (long long)blockIdx.x * (kmax + 1), N, dim, eps, kmax, S + blockIdx.x, red);
}

// ---------------------------------------------------------------------------------------------- host state
// One mutex serialises the entry points (they only enqueue work, so it is held for microseconds).  Settings are
// process-wide; everything that lives on a device (cached tile lists, events, the host path's buffers) is kept per
// CUDA device ordinal and looked up from cudaGetDevice() on every call, so a process may drive several GPUs.
// Cached device objects are created on first use and released ONLY by csg_shutdown(): a CUDA graph that captured a
// csg_action call keeps pointing at valid memory however many other sizes are run in between.
constexpr int TIMING_RING = 64;
constexpr int PROGRESS_RING = 64;
constexpr int MAX_DEVICES = 64;
constexpr int OCC_RING = 32;

struct TileList {                       // tile schedule of one (N, shard, nshards) on the device; nshards = -batch for a batch of sets
    long long N;
    int shard, nshards;
    int2* d;
    int n;
};
struct ChunkTiles {                     // the same tiles ordered by when the host-matrix pipeline makes them runnable
    long long N;
    int2* d;                            // tiles, sorted by need (stable: deepest first / patch order inside a step)
    int* d_need;                        // per tile: copy steps that must have completed before it may start
    int n;
    std::vector<int> off;               // tiles [off[s], off[s+1]) become runnable when copy step s completes
    std::vector<long long> row_begin, row_end;   // rows copied by step s
};
struct BitsMap {                        // TMA descriptor of a relation matrix (passed to the kernel by value)
    const void* ptr;
    long long N;                        // rows of the view (batch x N for a batch of sets)
    long long stride;
    int kind;
    CUtensorMap map;
};

struct Device {
    int ordinal = -1;
    int sm_count = 0;
    bool attr_set = false;
    int wait_clusters = -1;             // cudaOccupancyMaxActiveClusters of the WAIT instantiation (throttle needs all resident)
    std::vector<TileList> tiles;
    std::vector<ChunkTiles*> chunk_tiles;
    std::vector<BitsMap> maps;          // small ring, oldest replaced
    size_t maps_next = 0;
    // ring of event pairs around the interval kernel of the latest TIMING_RING timed calls
    cudaEvent_t ev0[TIMING_RING] = {}, ev1[TIMING_RING] = {};
    long long timed_calls = 0;
    unsigned int* d_progress = nullptr; // PROGRESS_RING finished-tile counters, one per launch in flight (drift throttle)
    std::map<cudaStream_t, BitsetFusedWs*> fused_ws;   // fused small-N launch: one zeroed workspace per stream
    unsigned int* d_landed = nullptr;   // chunks of the host matrix delivered so far (gate of csg_action_host)
    // block-occupancy bitmaps (occupancy_kernel.cuh), one per launch in flight; a slot that is too small for a later N is
    // replaced and the old buffer kept until csg_shutdown (a launch or a captured graph may still read it)
    uint32_t* d_occ[OCC_RING] = {};
    size_t d_occ_words[OCC_RING] = {};
    std::vector<uint32_t*> occ_retired;
    long long occ_next = 0;
    // end-to-end (host buffer) path
    cudaStream_t host_stream = nullptr, copy_stream = nullptr, occ_stream = nullptr;
    uint64_t* d_bits = nullptr;
    size_t d_bits_bytes = 0;
    long long* d_counts = nullptr;
    size_t d_counts_bytes = 0;
    double* d_S = nullptr;
    double* d_coords = nullptr;
    size_t d_coords_bytes = 0;
    std::vector<cudaEvent_t> chunk_ev;
    // events around the latest timed linking kernel
    cudaEvent_t link_ev0 = nullptr, link_ev1 = nullptr;
    bool link_timed = false;
};

struct Global {
    std::mutex mu;
    int variant = CSG_VARIANT_AUTO;
    int throttle = CSG_THROTTLE_AUTO;
    int sparse = CSG_SPARSE_AUTO;
    int host_pipeline = CSG_HOST_PIPELINE_AUTO;
    bool timing = false;
    int debug = 0;                      // ablation bits; only the -DCSG_ABLATE build can set it
    long long launches = 0;
    char cuda_msg[256] = "no CUDA error recorded";
    void* encode_tiled = nullptr;       // cuTensorMapEncodeTiled
    void* write_value32 = nullptr;      // cuStreamWriteValue32
    bool write_value32_tried = false;
    Device* dev[MAX_DEVICES] = {};
};
static Global g;

static int cuda_fail(cudaError_t e, const char* what) {
    snprintf(g.cuda_msg, sizeof(g.cuda_msg), "%s: %s", what, cudaGetErrorString(e));
    cudaGetLastError();  // clear the sticky-less error state
    return CSG_E_CUDA;
}
#define CSG_CUDA(call)                                   \
    do {                                                 \
        cudaError_t e_ = (call);                         \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
    } while (0)

// State of the current CUDA device (created on first use).
static int current_device(Device** out) {
    int ord = 0;
    CSG_CUDA(cudaGetDevice(&ord));
    if (ord < 0 || ord >= MAX_DEVICES) {
        snprintf(g.cuda_msg, sizeof(g.cuda_msg), "device ordinal %d out of range", ord);
        return CSG_E_CUDA;
    }
    if (!g.dev[ord]) {
        cudaDeviceProp prop;
        CSG_CUDA(cudaGetDeviceProperties(&prop, ord));
        if (prop.major != 10) {
            snprintf(g.cuda_msg, sizeof(g.cuda_msg), "device is sm_%d%d; libcsg is built for sm_100a only", prop.major,
                     prop.minor);
            return CSG_E_CUDA;
        }
        Device* d = new Device;
        d->ordinal = ord;
        d->sm_count = prop.multiProcessorCount;
        g.dev[ord] = d;
    }
    *out = g.dev[ord];
    return CSG_OK;
}

// Measured on B200 (CUDA-event ms of the interval kernel, 2D sets): N = 1024: bitset 0.0127 / fp4 0.0126;
// 1536: 0.0268 / 0.0151; 2048: 0.0378 / 0.0149; 4096: 0.158 / 0.021.  One set: fp4 above 1024.  A batch shares one
// bitset launch over all its sets, which beats back-to-back fp4 launches until the sets are 2048 and larger.
static int effective_variant(long long N) {
    if (g.variant != CSG_VARIANT_AUTO) return g.variant;
    return N > 1024 ? CSG_VARIANT_TENSOR_FP4 : CSG_VARIANT_BITSET;
}
// A batch: the tensor variant works through all sets in one persistent launch (ensure_batch_tiles).  Measured on B200, 64
// sets of 2D orders, ms per call, bitset launch / fp4 launch: N = 64: 0.0204 / 0.0202 (both launch-bound); 200: 0.0246 /
// 0.0204; 300: 0.0336 / 0.0206; 512: 0.0715 / 0.0201; 1024: 0.2896 / 0.0357; 2048: 1.559 / 0.109; 4096 sets of N = 1024:
// 11.54 / 1.448 ms.  So only sets that fit in one half-filled tile stay with the bitset kernel.
constexpr long long BATCH_TENSOR_MIN_N = 129;
constexpr long long BATCH_MAX_TILES = 4LL << 20;      // entries of one batch tile list (32 MiB)
static int effective_batch_variant(long long N) {
    if (g.variant != CSG_VARIANT_AUTO) return g.variant;
    return N >= BATCH_TENSOR_MIN_N ? CSG_VARIANT_TENSOR_FP4 : CSG_VARIANT_BITSET;
}

// Tile schedule of the tensor variant (pure host logic; exported as csg_tile_schedule).  Tiles (I, J) in
// 256-row blocks, I <= J; the K-depth of a tile is J-I+1 blocks, so the upper triangle is a triangular workload.
//   * matrix within L2 (<= TILE_L2_BYTES): tiles sorted by depth, longest first; shard s takes every nshards-th.
//   * larger: tiles grouped in patches of PATCH_H x PATCH_W blocks (about one tile per persistent cluster), patches
//     sorted by their deepest tile, tiles inside a patch by depth.  The clusters of one round then stream the same
//     PATCH_H + PATCH_W row blocks at about the same K, so each row segment comes from HBM once per patch and from
//     L2 for the other tiles of the patch; whole patches are dealt to the shards, least-loaded shard first.
// Longest first keeps the tail short; the kernel deals consecutive tiles boustrophedon to its persistent clusters.
constexpr long long TILE_L2_BYTES = 48LL << 20;
constexpr int PATCH_H = 8, PATCH_W = 9;

static void build_tile_schedule(long long N, int shard, int nshards, std::vector<int2>& out) {
    out.clear();
    const int nB = (int)((N + TC_T - 1) / TC_T);
    const long long bytes = N * (long long)(4 * ((N + 255) / 256)) * 8;
    if (bytes <= TILE_L2_BYTES) {
        long long t = 0;
        for (int d = nB - 1; d >= 0; --d)
            for (int I = 0; I + d < nB; ++I, ++t)
                if (t % nshards == shard) out.push_back(make_int2(I, I + d));
        return;
    }
    struct Patch { int depth, p, q; };
    std::vector<Patch> patches;
    const int nP = (nB + PATCH_H - 1) / PATCH_H, nQ = (nB + PATCH_W - 1) / PATCH_W;
    for (int p = 0; p < nP; ++p)
        for (int q = 0; q < nQ; ++q) {
            const int Ilo = p * PATCH_H, Jhi = std::min(nB, (q + 1) * PATCH_W) - 1;
            if (Jhi >= Ilo) patches.push_back({Jhi - Ilo, p, q});
        }
    std::stable_sort(patches.begin(), patches.end(), [](const Patch& a, const Patch& b) { return a.depth > b.depth; });
    // patches go, deepest first, to the shard with the least work so far (work = sum of K-depths; every rank
    // computes the same assignment)
    std::vector<long long> load(nshards, 0);
    std::vector<int2> in_patch;
    for (size_t k = 0; k < patches.size(); ++k) {
        const Patch& pt = patches[k];
        in_patch.clear();
        long long work = 0;
        for (int I = pt.p * PATCH_H; I < std::min(nB, (pt.p + 1) * PATCH_H); ++I)
            for (int J = std::max(I, pt.q * PATCH_W); J < std::min(nB, (pt.q + 1) * PATCH_W); ++J) {
                in_patch.push_back(make_int2(I, J));
                work += J - I + 1;
            }
        const int owner = (int)(std::min_element(load.begin(), load.end()) - load.begin());
        load[owner] += work;
        if (owner != shard) continue;
        std::stable_sort(in_patch.begin(), in_patch.end(),
                         [](const int2& a, const int2& b) { return a.y - a.x > b.y - b.x; });
        out.insert(out.end(), in_patch.begin(), in_patch.end());
    }
}

// Device copy of a shard's tile list.  Built on the first call for that (N, shard, nshards) with one blocking copy;
// afterwards a lookup.  Entries stay until csg_shutdown (at most 4 MiB each, N = 262144), so a captured CUDA graph or a
// launch in flight on another stream never sees its tile list freed or overwritten.
static int ensure_tiles(Device* D, long long N, int shard, int nshards, const TileList** out) {
    for (const TileList& t : D->tiles)
        if (t.N == N && t.shard == shard && t.nshards == nshards) {
            *out = &t;
            return CSG_OK;
        }
    std::vector<int2> h;
    build_tile_schedule(N, shard, nshards, h);
    TileList t{N, shard, nshards, nullptr, (int)h.size()};
    CSG_CUDA(cudaMalloc(&t.d, std::max<size_t>(1, h.size()) * sizeof(int2)));
    if (!h.empty()) CSG_CUDA(cudaMemcpy(t.d, h.data(), h.size() * sizeof(int2), cudaMemcpyHostToDevice));
    D->tiles.push_back(t);
    *out = &D->tiles.back();
    return CSG_OK;
}

// Tile list of a batch of `batch` sets of N elements (csg_action_batch on the tensor cores): all sets' tiles in one
// list, deepest first across the whole batch, the set index packed into the first coordinate (TC_SET_SHIFT), so that
// ONE persistent launch works through the batch without a tail per set.  Cached like the single-set lists.
static int ensure_batch_tiles(Device* D, long long N, int batch, const TileList** out) {
    for (const TileList& t : D->tiles)
        if (t.N == N && t.shard == 0 && t.nshards == -batch) {
            *out = &t;
            return CSG_OK;
        }
    const int nB = (int)((N + TC_T - 1) / TC_T);
    std::vector<int2> h;
    h.reserve((size_t)batch * nB * (nB + 1) / 2);
    for (int d = nB - 1; d >= 0; --d)
        for (int b = 0; b < batch; ++b)
            for (int I = 0; I + d < nB; ++I) h.push_back(make_int2(I | (b << TC_SET_SHIFT), I + d));
    TileList t{N, 0, -batch, nullptr, (int)h.size()};
    CSG_CUDA(cudaMalloc(&t.d, std::max<size_t>(1, h.size()) * sizeof(int2)));
    if (!h.empty()) CSG_CUDA(cudaMemcpy(t.d, h.data(), h.size() * sizeof(int2), cudaMemcpyHostToDevice));
    D->tiles.push_back(t);
    *out = &D->tiles.back();
    return CSG_OK;
}

// 2D byte view of the packed relation matrix for the TMA warp of the tensor variants: dim0 = stride*8 bytes of a
// row, dim1 = N rows; box = 32 (int8) or 64 (fp4) bytes x 128 rows with the matching 32/64-byte swizzle
// (conflict-free 16-byte reads by the producers); rows >= N and bytes beyond the row are zero-filled by the hardware.
// The descriptor is a kernel parameter (copied at launch), so this cache is host memory only.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
typedef CUresult (*WriteValue32Fn)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
constexpr size_t MAPS_CACHED = 16;

static int ensure_bits_map(Device* D, int kind, const uint64_t* rel_bits, long long N, long long stride_words,
                           const CUtensorMap** out) {
    for (const BitsMap& m : D->maps)
        if (m.ptr == rel_bits && m.N == N && m.stride == stride_words && m.kind == kind) {
            *out = &m.map;
            return CSG_OK;
        }
    if (!g.encode_tiled) {
        cudaDriverEntryPointQueryResult qres;
        CSG_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &g.encode_tiled, cudaEnableDefault, &qres));
        if (qres != cudaDriverEntryPointSuccess || !g.encode_tiled) {
            snprintf(g.cuda_msg, sizeof(g.cuda_msg), "cuTensorMapEncodeTiled not available from the driver");
            g.encode_tiled = nullptr;
            return CSG_E_CUDA;
        }
    }
    BitsMap m{rel_bits, N, stride_words, kind, {}};
    const int row_bytes = kind == KIND_FP4 ? TcTraits<KIND_FP4>::BITS_ROW_BYTES : TcTraits<KIND_I8>::BITS_ROW_BYTES;
    const cuuint64_t dims[2] = {(cuuint64_t)stride_words * 8, (cuuint64_t)N};
    const cuuint64_t strides[1] = {(cuuint64_t)stride_words * 8};
    const cuuint32_t box[2] = {(cuuint32_t)row_bytes, (cuuint32_t)TC_BITS_BOX_ROWS};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = reinterpret_cast<EncodeTiledFn>(g.encode_tiled)(
        &m.map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint64_t*>(rel_bits), dims, strides, box, estr,
        CU_TENSOR_MAP_INTERLEAVE_NONE, kind == KIND_FP4 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_32B,
        CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g.cuda_msg, sizeof(g.cuda_msg), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        return CSG_E_CUDA;
    }
    if (D->maps.size() < MAPS_CACHED) {
        D->maps.push_back(m);
        *out = &D->maps.back().map;
    } else {
        D->maps[D->maps_next] = m;
        *out = &D->maps[D->maps_next].map;
        D->maps_next = (D->maps_next + 1) % MAPS_CACHED;
    }
    return CSG_OK;
}

static int validate(const void* rel_bits, long long N, int dim, double eps, int kmax, const void* counts,
                    const void* S) {
    if (!rel_bits || !counts || !S) return CSG_E_NULL;
    if (N < 1 || N > CSG_MAX_N) return CSG_E_SIZE;
    if (dim != 2 && dim != 4) return CSG_E_DIM;
    if (!(eps > 0.0 && eps <= 1.0)) return CSG_E_EPS;  // also rejects NaN
    if (kmax < 0 || kmax > CSG_MAX_KMAX) return CSG_E_KMAX;
    if (eps == 1.0 && kmax < (dim == 2 ? 2 : 3)) return CSG_E_KMAX;
    return CSG_OK;
}

#ifdef CSG_ABLATE
constexpr int FP4_EXTRA = TCF_ABLATE;   // the ablation build's fp4 kernel carries the dbg switches (wrong counts when set)
#else
constexpr int FP4_EXTRA = 0;
#endif

// Dynamic shared memory opt-in of the tensor kernels and the occupancy of the instantiation that may wait.
static int ensure_tensor_ready(Device* D) {
    if (D->attr_set) return CSG_OK;
    const int s8 = TcTraits<KIND_I8>::smem_bytes(TC_HIST_WHOLE), s4 = TcTraits<KIND_FP4>::smem_bytes(TC_HIST_WHOLE);   // the most a launch may ask for
#define CSG_OPT_IN(kernel, bytes) CSG_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))
    CSG_OPT_IN((tensor_action_kernel<KIND_I8, 7>), s8);
    CSG_OPT_IN((tensor_action_kernel<KIND_I8, 6>), s8);
    CSG_OPT_IN((tensor_action_kernel<KIND_I8, 5>), s8);
    CSG_OPT_IN((tensor_action_kernel<KIND_I8, 4>), s8);
    CSG_OPT_IN((tensor_action_kernel<KIND_I8, 7, TCF_DUMP>), s8);
    CSG_OPT_IN((tensor_action_kernel<KIND_I8, 6, TCF_DUMP>), s8);
    CSG_OPT_IN((tensor_action_kernel<KIND_I8, 5, TCF_DUMP>), s8);
    CSG_OPT_IN((tensor_action_kernel<KIND_I8, 4, TCF_DUMP>), s8);
    CSG_OPT_IN((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA>), s4);
    CSG_OPT_IN((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_WAIT>), s4);
    CSG_OPT_IN((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_SPARSE>), s4);
    CSG_OPT_IN((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_SPARSE | TCF_WAIT>), s4);
    CSG_OPT_IN((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_GATE>), s4);
    CSG_OPT_IN((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_GATE | TCF_SPARSE>), s4);
    CSG_OPT_IN((tensor_action_kernel<KIND_FP4, 0, TCF_DUMP | TCF_SPARSE>), s4);
    CSG_OPT_IN((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_BATCH>), s4);
    CSG_OPT_IN((tensor_action_kernel<KIND_I8, 7, TCF_BATCH>), s8);
    CSG_OPT_IN((tensor_peak_kernel<KIND_FP4>), s4);
    CSG_OPT_IN((tensor_peak_kernel<KIND_I8>), s8);
#undef CSG_OPT_IN
    // Kernels that the host-matrix pipeline launches WHILE its gated interval kernel is already running (and waiting for
    // the chunks the host is still enqueueing) must be loaded beforehand: with CUDA's lazy module loading the first
    // launch of a kernel loads it, loading may synchronise the context, and that would wait for the gated kernel, which
    // waits for the host -- csg_action_host as the FIRST call of a process hung exactly there.  cudaFuncGetAttributes
    // forces the load.
    {
        cudaFuncAttributes fa;
        CSG_CUDA(cudaFuncGetAttributes(&fa, occupancy_kernel));
        CSG_CUDA(cudaFuncGetAttributes(&fa, finish_action_kernel));
    }
    // The drift throttle makes clusters wait for tiles finished by OTHER clusters, which is only safe when the whole
    // grid is resident at once: ask the runtime how many CTA pairs of that instantiation fit on the device right now.
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * (D->sm_count / 2));
    cfg.blockDim = dim3(TC_THREADS);
    cfg.dynamicSmemBytes = s4;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = 2;
    attr.val.clusterDim.y = 1;
    attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_SPARSE | TCF_WAIT>, &cfg) != cudaSuccess) {
        cudaGetLastError();
        nclusters = 0;
    }
    D->wait_clusters = nclusters;
    D->attr_set = true;
    return CSG_OK;
}

// One launch of the tensor kernel over a tile list (counts are added to, not zeroed).  landed / tile_need: gate of
// the host-matrix path (NULL when the matrix is resident); dump: csg_tile_interval_sizes (NULL otherwise).
// batch > 1: rel_bits holds `batch` matrices back to back and counts `batch` histograms of kmax + 1 bins (d_tiles from
// ensure_batch_tiles).
static int launch_tensor(Device* D, int kind, const uint64_t* rel_bits, long long N, long long stride, int kmax,
                         long long* counts, const int2* d_tiles, int ntiles, const unsigned int* landed,
                         const int* tile_need, int* dump, const uint32_t* occ, cudaStream_t stream, int batch = 1) {
    int rc = ensure_tensor_ready(D);
    if (rc) return rc;
    const CUtensorMap* map = nullptr;
    const int counts_stride = batch > 1 ? kmax + 1 : 0;
    rc = ensure_bits_map(D, kind, rel_bits, N * batch, stride, &map);
    if (rc) return rc;
    // One CTA pair per SM pair.  The gated launch of the host-matrix pipeline with the block-sparse sweep leaves one SM
    // pair free: it waits for occupancy kernels that are launched while it runs, and those must find an SM (next to a
    // CTA of this kernel there is no room: 18 warps x 96 registers fill two of the four register files of an SM).
    const int clusters = std::max(1, D->sm_count / 2 - ((landed && occ) ? 1 : 0));
    const int grid = 2 * std::max(1, std::min(ntiles, clusters));
    // Drift throttle (tensor_kernel.cuh, TC_MAX_LEAD): fewer DRAM reads, so less power.  Measured (round 2 kernel):
    // config 4 (N = 262144, 8 GiB, full histogram) 942 -> 847 ms; config 3 (N = 131072, 2 GiB), where the kernel now
    // runs into the 1 kW power cap: a single launch 88.5 either way, twelve back to back 89.9 (drifting up to 92) ->
    // 88.85 ms (steady); config 2 (512 MiB, no power cap) 12.02 -> 12.20 ms.  So CSG_THROTTLE_AUTO switches it on for
    // matrices above 1 GiB -- and in every mode only if the runtime says that the whole grid can be resident at once
    // (the wait is bounded in the kernel, too).
    unsigned int* progress = nullptr;
    const bool big = N * stride * 8 > (1LL << 30) && ntiles > 16 * (grid / 2);
    const bool want = g.throttle == CSG_THROTTLE_ON ? ntiles > grid / 2 : (g.throttle == CSG_THROTTLE_AUTO && big);
    if (kind == KIND_FP4 && dump == nullptr && want && D->wait_clusters >= grid / 2) {
        // a ring of counters, one per launch, so that launches in flight on different streams do not share one
        if (!D->d_progress) CSG_CUDA(cudaMalloc(&D->d_progress, PROGRESS_RING * sizeof(unsigned int)));
        progress = D->d_progress + (g.launches % PROGRESS_RING);
        CSG_CUDA(cudaMemsetAsync(progress, 0, sizeof(unsigned int), stream));
    }
    unsigned long long* c64 = reinterpret_cast<unsigned long long*>(counts);
    // private histogram: the large one only for launches that can reach bins beyond the small one (tensor_kernel.cuh: TC_HIST)
    const long long kcap = std::min<long long>(kmax, std::max<long long>(N - 2, 0));
    const int hist_bins = (dump == nullptr && batch == 1 && kcap >= TC_HIST) ? TC_HIST_WHOLE : TC_HIST;
    const int s8 = TcTraits<KIND_I8>::smem_bytes(hist_bins), s4 = TcTraits<KIND_FP4>::smem_bytes(hist_bins);
#define CSG_LAUNCH(KERNEL, SMEM) \
    KERNEL<<<grid, TC_THREADS, SMEM, stream>>>(*map, rel_bits, N, stride, kmax, c64, d_tiles, ntiles, g.debug, progress, landed, tile_need, dump, occ, occ_stride_words(N), counts_stride, hist_bins)
    // int8: operand bit TB: the accumulator holds n_ij << 2TB and n_ij <= N-2, so TB is the largest with
    // (N-2) << 2TB < 2^31; TB = 7 turns every unpack shift into a left shift (FMA pipe).
    const int tb = N - 2 < (1LL << 17) ? 7 : N - 2 < (1LL << 19) ? 6 : N - 2 < (1LL << 21) ? 5 : 4;
    if (kind == KIND_FP4) {
        // one instantiation per combination in use, so that a launch carries only the code it needs (tensor_kernel.cuh)
        if (batch > 1) CSG_LAUNCH((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_BATCH>), s4);
        else if (dump) CSG_LAUNCH((tensor_action_kernel<KIND_FP4, 0, TCF_DUMP | TCF_SPARSE>), s4);
        else if (landed && occ) CSG_LAUNCH((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_GATE | TCF_SPARSE>), s4);
        else if (landed) CSG_LAUNCH((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_GATE>), s4);
        else if (progress && occ) CSG_LAUNCH((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_SPARSE | TCF_WAIT>), s4);
        else if (progress) CSG_LAUNCH((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_WAIT>), s4);
        else if (occ) CSG_LAUNCH((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA | TCF_SPARSE>), s4);
        else CSG_LAUNCH((tensor_action_kernel<KIND_FP4, 0, FP4_EXTRA>), s4);
    } else if (batch > 1) {
        if (tb != 7) {      // batches are sets within L2 (N < 2^17), for which the int8 kind always has TB = 7
            snprintf(g.cuda_msg, sizeof(g.cuda_msg), "batched int8 launch with N = %lld", N);
            return CSG_E_CUDA;
        }
        CSG_LAUNCH((tensor_action_kernel<KIND_I8, 7, TCF_BATCH>), s8);
    } else if (dump) {
        if (tb == 7) CSG_LAUNCH((tensor_action_kernel<KIND_I8, 7, TCF_DUMP>), s8);
        else if (tb == 6) CSG_LAUNCH((tensor_action_kernel<KIND_I8, 6, TCF_DUMP>), s8);
        else if (tb == 5) CSG_LAUNCH((tensor_action_kernel<KIND_I8, 5, TCF_DUMP>), s8);
        else CSG_LAUNCH((tensor_action_kernel<KIND_I8, 4, TCF_DUMP>), s8);
    } else {
        if (tb == 7) CSG_LAUNCH((tensor_action_kernel<KIND_I8, 7>), s8);
        else if (tb == 6) CSG_LAUNCH((tensor_action_kernel<KIND_I8, 6>), s8);
        else if (tb == 5) CSG_LAUNCH((tensor_action_kernel<KIND_I8, 5>), s8);
        else CSG_LAUNCH((tensor_action_kernel<KIND_I8, 4>), s8);
    }
#undef CSG_LAUNCH
    CSG_CUDA(cudaGetLastError());
    ++g.launches;
    return CSG_OK;
}

// Block-sparse K sweep of the fp4 tensor kernel (occupancy_kernel.cuh): one pass over the matrix marks the empty
// 256 x 256 blocks, and the kernel skips every two-stage group whose U or L blocks are empty.  Measured at config 3 (4D,
// N = 131072): 10.8 % of the groups are dead, 88.5 -> 81.8 ms.  A 1+1 set (flat or de Sitter) has no empty block: there
// the pass and the mask loop cost 2 % (de Sitter N = 131072: 94.0 -> 96.0 ms).  So CSG_SPARSE_AUTO switches it on for
// matrices of 96 MiB and more unless the caller says dim = 2 (csg_action_partial has no dim: on); ON: every fp4
// launch (tests).  *occ = nullptr when the sweep stays dense.
// The threshold: 3+1 sprinklings have 11-12 % dead groups from N = 16384 on (5 % at 8192), but the occupancy pass is one
// more dependent launch: measured dense / sparse ms at N = 8192: 0.047 / 0.063, 16384 (32 MiB): 0.234 / 0.244, 24576
// (72 MiB): 0.706 / 0.708, 32768 (128 MiB): 1.603 / 1.551, 49152 (288 MiB): 4.94 / 4.64, 65536: 11.6 / 10.7.
constexpr long long SPARSE_MIN_BYTES = 96LL << 20;

// The occupancy map of the next launch (one of OCC_RING buffers), or *occ = nullptr when the sweep stays dense.
static int occupancy_buffer(Device* D, int kind, long long N, long long stride, int dim_hint, uint32_t** occ) {
    *occ = nullptr;
    if (kind != KIND_FP4 || g.sparse == CSG_SPARSE_OFF) return CSG_OK;
    if (g.sparse == CSG_SPARSE_AUTO && (N * stride * 8 < SPARSE_MIN_BYTES || dim_hint == 2)) return CSG_OK;
    const int nB = (int)((N + TC_T - 1) / TC_T);
    const size_t words = (size_t)nB * occ_stride_words(N);
    const int slot = (int)(D->occ_next++ % OCC_RING);
    if (D->d_occ_words[slot] < words) {
        // the whole ring at once, so that after ONE warm-up call of a size no later call of that size allocates (a call
        // that is being captured into a CUDA graph must not)
        for (int k = 0; k < OCC_RING; ++k) {
            if (D->d_occ_words[k] >= words) continue;
            if (D->d_occ[k]) D->occ_retired.push_back(D->d_occ[k]);
            D->d_occ[k] = nullptr;
            D->d_occ_words[k] = 0;
            CSG_CUDA(cudaMalloc(&D->d_occ[k], words * sizeof(uint32_t)));
            D->d_occ_words[k] = words;
        }
    }
    *occ = D->d_occ[slot];
    return CSG_OK;
}

// Marks row blocks [block0, block0 + nblocks) of the map.
static int occupancy_launch(const uint64_t* rel_bits, long long N, long long stride, uint32_t* occ, int block0, int nblocks,
                            cudaStream_t stream) {
    const int ostride = occ_stride_words(N);
    occupancy_kernel<<<dim3(ostride / OCC_WORDS_PER_CTA, nblocks), OCC_THREADS, 0, stream>>>(rel_bits, N, stride, occ, ostride, block0);
    CSG_CUDA(cudaGetLastError());
    ++g.launches;
    return CSG_OK;
}

static int occupancy_pass(Device* D, int kind, const uint64_t* rel_bits, long long N, long long stride, int dim_hint,
                          const uint32_t** occ, cudaStream_t stream) {
    uint32_t* buf = nullptr;
    *occ = nullptr;
    int rc = occupancy_buffer(D, kind, N, stride, dim_hint, &buf);
    if (rc || !buf) return rc;
    if ((rc = occupancy_launch(rel_bits, N, stride, buf, 0, (int)((N + TC_T - 1) / TC_T), stream))) return rc;
    *occ = buf;
    return CSG_OK;
}

// Interval kernel over the tiles of one shard: counts (kmax+1 int64, overwritten) <- this shard's abundances.
// dim_hint: the caller's dim (2 or 4) or 0 when the entry point has none; only steers CSG_SPARSE_AUTO.
static int interval_device(Device* D, const uint64_t* rel_bits, long long N, int kmax, int shard, int nshards, int dim_hint,
                           long long* counts, cudaStream_t stream) {
    const long long stride = csg_row_stride_words(N);
    CSG_CUDA(cudaMemsetAsync(counts, 0, (size_t)(kmax + 1) * sizeof(long long), stream));
    const int variant = effective_variant(N);
    const bool tensor = variant == CSG_VARIANT_TENSOR || variant == CSG_VARIANT_TENSOR_FP4;
    const int kind = variant == CSG_VARIANT_TENSOR_FP4 ? KIND_FP4 : KIND_I8;
    const TileList* tl = nullptr;
    int rc;
    if (tensor) {
        rc = ensure_tiles(D, N, shard, nshards, &tl);
        if (rc) return rc;
    }
    const int slot = (int)(D->timed_calls % TIMING_RING);
    if (g.timing) {
        if (!D->ev0[slot]) {
            CSG_CUDA(cudaEventCreate(&D->ev0[slot]));
            CSG_CUDA(cudaEventCreate(&D->ev1[slot]));
        }
        CSG_CUDA(cudaEventRecord(D->ev0[slot], stream));
    }
    if (tensor) {
        const uint32_t* occ = nullptr;
        if ((rc = occupancy_pass(D, kind, rel_bits, N, stride, dim_hint, &occ, stream))) return rc;
        rc = launch_tensor(D, kind, rel_bits, N, stride, kmax, counts, tl->d, tl->n, nullptr, nullptr, nullptr, occ, stream);
        if (rc) return rc;
    } else {
        const long long nb = (N + BS_T - 1) / BS_T;
        const long long ntiles = nb * (nb + 1) / 2;
        const long long mine = (ntiles - shard + nshards - 1) / nshards;   // tiles t = shard (mod nshards)
        const int grid = (int)std::max<long long>(1, std::min<long long>(mine, (long long)D->sm_count * 2));
        bitset_action_kernel<<<grid, BS_THREADS, 0, stream>>>(reinterpret_cast<const uint32_t*>(rel_bits), N,
                                                               stride * 2, kmax,
                                                               reinterpret_cast<unsigned long long*>(counts), nb,
                                                               ntiles, shard, nshards, 0, 0, nullptr, 0, 1.0, nullptr);
        CSG_CUDA(cudaGetLastError());
        ++g.launches;
    }
    if (g.timing) {
        CSG_CUDA(cudaEventRecord(D->ev1[slot], stream));
        ++D->timed_calls;
    }
    return CSG_OK;
}

static int finish_device(const long long* counts, long long N, int dim, double eps, int kmax, double* S,
                         cudaStream_t stream) {
    finish_action_kernel<<<1, FIN_THREADS, 0, stream>>>(counts, N, dim, eps, kmax, S);
    CSG_CUDA(cudaGetLastError());
    ++g.launches;
    return CSG_OK;
}

// Small sets on the bitset variant: memset, interval kernel and finishing kernel in ONE launch (bitset_kernel.cuh).
// The workspace is per stream, so launches that share it run one after the other; a stream that is being captured
// (the graph may later run next to eager launches of its source stream) and the per-thread default stream (one
// handle, many streams) take the three-node path instead.
static bool fused_small_ok(long long N, int kmax, cudaStream_t stream) {
    if (effective_variant(N) != CSG_VARIANT_BITSET || kmax >= BS_FUSED_BINS || stream == cudaStreamPerThread) return false;
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &st) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return st == cudaStreamCaptureStatusNone;
}

static int action_fused_small(Device* D, const uint64_t* rel_bits, long long N, int dim, double eps, int kmax,
                              long long* counts, double* S, cudaStream_t stream) {
    BitsetFusedWs*& ws = D->fused_ws[stream];
    if (!ws) {
        CSG_CUDA(cudaMalloc(&ws, sizeof(BitsetFusedWs)));
        CSG_CUDA(cudaMemset(ws, 0, sizeof(BitsetFusedWs)));
    }
    const long long stride = csg_row_stride_words(N);
    const long long nb = (N + BS_T - 1) / BS_T;
    const long long ntiles = nb * (nb + 1) / 2;
    const int grid = (int)std::max<long long>(1, std::min<long long>(ntiles, (long long)D->sm_count * 2));
    const int slot = (int)(D->timed_calls % TIMING_RING);
    if (g.timing) {
        if (!D->ev0[slot]) {
            CSG_CUDA(cudaEventCreate(&D->ev0[slot]));
            CSG_CUDA(cudaEventCreate(&D->ev1[slot]));
        }
        CSG_CUDA(cudaEventRecord(D->ev0[slot], stream));
    }
    bitset_action_kernel<<<grid, BS_THREADS, 0, stream>>>(reinterpret_cast<const uint32_t*>(rel_bits), N, stride * 2, kmax,
                                                           reinterpret_cast<unsigned long long*>(counts), nb, ntiles, 0, 1, 0,
                                                           0, ws, dim, eps, S);
    CSG_CUDA(cudaGetLastError());
    ++g.launches;
    if (g.timing) {
        CSG_CUDA(cudaEventRecord(D->ev1[slot], stream));
        ++D->timed_calls;
    }
    return CSG_OK;
}

static int action_device(Device* D, const uint64_t* rel_bits, long long N, int dim, double eps, int kmax,
                         long long* counts, double* S, cudaStream_t stream) {
    if (fused_small_ok(N, kmax, stream)) return action_fused_small(D, rel_bits, N, dim, eps, kmax, counts, S, stream);
    int rc = interval_device(D, rel_bits, N, kmax, 0, 1, dim, counts, stream);
    if (rc) return rc;
    return finish_device(counts, N, dim, eps, kmax, S, stream);
}

// Host matrix -> device in row chunks on a copy stream while the tiles already run (Sec. 2.2.5:
// overlap of transfers with compute).  A tile (I, J) reads the rows of blocks I and J only, so it is runnable as soon
// as the chunks holding those two blocks have landed.  The chunks are copied OUTSIDE-IN (first, last, second, ...):
// the first two chunks already make the deepest tiles of the triangle runnable, and after a fraction f of the copy
// 1.5 f^2 - 0.5 f^3 of the work is available instead of the f^3 of a front-to-back copy.  With the copy taking T_c and
// the kernel T_k the transfer then costs max_f [T_c f - T_k (1.5 f^2 - 0.5 f^3)]: about 3 ms at N = 131072 (41 ms of
// PCIe copy, 91 ms of kernel) against 10.6 ms front to back (measured 10.9) and 41 ms without overlap.
// The tile list is sorted by the copy step that makes a tile runnable (stable, so inside a step the schedule's
// deepest-first patch order survives).  Two ways to run it:
//   gated (fp4 kind, when the driver offers cuStreamWriteValue32): ONE persistent launch; after every chunk the copy
//     stream publishes the number of chunks delivered and the TMA thread of a cluster waits for the count its next
//     tile needs -- no launch tails between chunks;
//   chunked launches (int8 kind, or no stream memory operations): one launch per copy step behind an event.
// Tensor variants and large matrices only.
constexpr int HOST_CHUNKS = 64;
constexpr long long HOST_PIPELINE_MIN_BYTES = 32LL << 20;

static int ensure_chunk_tiles(Device* D, long long N, const ChunkTiles** out) {
    for (const ChunkTiles* c : D->chunk_tiles)
        if (c->N == N) {
            *out = c;
            return CSG_OK;
        }
    const int nB = (int)((N + TC_T - 1) / TC_T);
    const int blocks_per_chunk = (nB + HOST_CHUNKS - 1) / HOST_CHUNKS;
    const int nchunks = (nB + blocks_per_chunk - 1) / blocks_per_chunk;
    // copy order outside-in: chunk 0, nchunks-1, 1, nchunks-2, ...; step_of[c] = position of chunk c in that order
    std::vector<int> step_of(nchunks);
    ChunkTiles* c = new ChunkTiles;
    c->N = N;
    c->d = nullptr;
    c->d_need = nullptr;
    for (int s = 0, lo = 0, hi = nchunks - 1; s < nchunks; ++s) {
        const int chunk = (s & 1) ? hi-- : lo++;
        step_of[chunk] = s;
        c->row_begin.push_back((long long)chunk * blocks_per_chunk * TC_T);
        c->row_end.push_back(std::min<long long>(N, (long long)(chunk + 1) * blocks_per_chunk * TC_T));
    }
    std::vector<int2> all;
    build_tile_schedule(N, 0, 1, all);
    std::vector<std::vector<int2>> per(nchunks);
    for (const int2& t : all)       // runnable after the later of its two chunks; keeps the schedule's order inside a step
        per[std::max(step_of[t.x / blocks_per_chunk], step_of[t.y / blocks_per_chunk])].push_back(t);
    std::vector<int2> flat;
    std::vector<int> need;
    c->off.assign(1, 0);
    for (int s = 0; s < nchunks; ++s) {
        flat.insert(flat.end(), per[s].begin(), per[s].end());
        need.insert(need.end(), per[s].size(), s + 1);
        c->off.push_back((int)flat.size());
    }
    c->n = (int)flat.size();
    cudaError_t e = cudaMalloc(&c->d, flat.size() * sizeof(int2));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_need, need.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(c->d, flat.data(), flat.size() * sizeof(int2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_need, need.data(), need.size() * sizeof(int), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        if (c->d) cudaFree(c->d);
        if (c->d_need) cudaFree(c->d_need);
        delete c;
        return cuda_fail(e, "tile list of the host pipeline");
    }
    while ((int)D->chunk_ev.size() < 2 * nchunks + 2) {
        cudaEvent_t ev;
        CSG_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        D->chunk_ev.push_back(ev);
    }
    D->chunk_tiles.push_back(c);
    *out = c;
    return CSG_OK;
}

static WriteValue32Fn stream_write_value32() {
    if (!g.write_value32_tried) {
        g.write_value32_tried = true;
        cudaDriverEntryPointQueryResult qres;
        void* fn = nullptr;
        if (cudaGetDriverEntryPoint("cuStreamWriteValue32", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            g.write_value32 = fn;
        else
            cudaGetLastError();
    }
    return reinterpret_cast<WriteValue32Fn>(g.write_value32);
}

// A gated launch waits inside the kernel for the chunk count; if feeding it fails half-way (a copy, an occupancy launch
// or a stream write returns an error) the count would never arrive and the caller's synchronize would hang.  The guard
// opens the gate on every early return: the launch then runs to its end on whatever has landed (the call returns the
// error, its counts are not used).
struct GateGuard {
    unsigned int* d_landed = nullptr;
    bool armed = false;
    ~GateGuard() {
        if (!armed) return;
        const unsigned int open = 0x7FFFFFFFu;
        cudaMemcpy(d_landed, &open, sizeof(open), cudaMemcpyHostToDevice);   // legacy default stream: does not wait for the non-blocking streams
        cudaGetLastError();
    }
};

static int interval_host_pipelined(Device* D, const uint64_t* rel_bits_host, uint64_t* d_bits, long long N, int kmax,
                                   int kind, int dim_hint, long long* counts, cudaStream_t stream) {
    const long long stride = csg_row_stride_words(N);
    const ChunkTiles* ct = nullptr;
    int rc = ensure_chunk_tiles(D, N, &ct);
    if (rc) return rc;
    if (!D->copy_stream) CSG_CUDA(cudaStreamCreateWithFlags(&D->copy_stream, cudaStreamNonBlocking));
    CSG_CUDA(cudaMemsetAsync(counts, 0, (size_t)(kmax + 1) * sizeof(long long), stream));
    const int nchunks = (int)ct->row_end.size();       // = copy steps
    cudaEvent_t ev_prev = D->chunk_ev[nchunks], ev_reset = D->chunk_ev[nchunks + 1];
    // the copies must not overtake work of an earlier call that still reads d_bits on `stream`
    CSG_CUDA(cudaEventRecord(ev_prev, stream));
    CSG_CUDA(cudaStreamWaitEvent(D->copy_stream, ev_prev, 0));
    // Block-sparse sweep: the row blocks of a chunk are marked (occupancy kernel) right behind the chunk's copy and BEFORE
    // the chunk is published, so the two occupancy rows a tile reads are complete when the tile may start.  The kernels
    // run on a stream of their own (behind an event per copy), so the copies stay back to back; that stream then
    // publishes the chunks.  A gated launch leaves them one SM pair (launch_tensor).
    uint32_t* occ = nullptr;
    if ((rc = occupancy_buffer(D, kind, N, stride, dim_hint, &occ))) return rc;
    if (occ && !D->occ_stream) CSG_CUDA(cudaStreamCreateWithFlags(&D->occ_stream, cudaStreamNonBlocking));
    cudaStream_t publish = occ ? D->occ_stream : D->copy_stream;
    WriteValue32Fn write32 = kind == KIND_FP4 && g.host_pipeline != CSG_HOST_PIPELINE_CHUNKED ? stream_write_value32() : nullptr;
    GateGuard gate;
    if (write32) {
        if (!D->d_landed) CSG_CUDA(cudaMalloc(&D->d_landed, sizeof(unsigned int)));
        // reset the gate, then ONE launch that starts at once and follows the copies
        if (write32(D->copy_stream, (CUdeviceptr)D->d_landed, 0u, 0) != CUDA_SUCCESS) {
            write32 = nullptr;                                 // no stream memory operations here: chunked launches
        } else {
            CSG_CUDA(cudaEventRecord(ev_reset, D->copy_stream));
            CSG_CUDA(cudaStreamWaitEvent(stream, ev_reset, 0));
            rc = launch_tensor(D, kind, d_bits, N, stride, kmax, counts, ct->d, ct->n, D->d_landed, ct->d_need, nullptr, occ, stream);
            if (rc) return rc;
            gate.d_landed = D->d_landed;
            gate.armed = true;
        }
    }
    for (int c = 0; c < nchunks; ++c) {
        const long long row0 = ct->row_begin[c], row1 = ct->row_end[c];
        CSG_CUDA(cudaMemcpyAsync(d_bits + row0 * stride, rel_bits_host + row0 * stride,
                                 (size_t)(row1 - row0) * stride * sizeof(uint64_t), cudaMemcpyHostToDevice, D->copy_stream));
        if (occ) {
            CSG_CUDA(cudaEventRecord(D->chunk_ev[nchunks + 2 + c], D->copy_stream));
            CSG_CUDA(cudaStreamWaitEvent(D->occ_stream, D->chunk_ev[nchunks + 2 + c], 0));
            const int b0 = (int)(row0 / TC_T), b1 = (int)((row1 + TC_T - 1) / TC_T);
            if ((rc = occupancy_launch(d_bits, N, stride, occ, b0, b1 - b0, D->occ_stream))) return rc;
        }
        if (write32) {
            if (write32(publish, (CUdeviceptr)D->d_landed, (cuuint32_t)(c + 1), 0) != CUDA_SUCCESS) {
                snprintf(g.cuda_msg, sizeof(g.cuda_msg), "cuStreamWriteValue32 failed while a gated launch is waiting");
                return CSG_E_CUDA;
            }
        } else {
            CSG_CUDA(cudaEventRecord(D->chunk_ev[c], publish));
            CSG_CUDA(cudaStreamWaitEvent(stream, D->chunk_ev[c], 0));
            const int nt = ct->off[c + 1] - ct->off[c];
            if (nt > 0) {
                rc = launch_tensor(D, kind, d_bits, N, stride, kmax, counts, ct->d + ct->off[c], nt, nullptr, nullptr, nullptr, occ, stream);
                if (rc) return rc;
            }
        }
    }
    gate.armed = false;                 // every chunk has been published (or nothing was gated)
    return CSG_OK;
}

static int geometry_dim(int geometry) { return geometry == CSG_GEOM_MINKOWSKI_4D ? 4 : 2; }

// Linking kernel on `stream`: every word of rel_bits (N rows x stride) is overwritten.
static int link_device(Device* D, const double* coords, long long N, int geometry, uint64_t* rel_bits,
                       cudaStream_t stream) {
    const long long stride = csg_row_stride_words(N);
    const int nB = (int)((N + LK_T - 1) / LK_T);
    const long long ntiles = (long long)nB * (nB + 1) / 2;
    if (g.timing) {
        if (!D->link_ev0) {
            CSG_CUDA(cudaEventCreate(&D->link_ev0));
            CSG_CUDA(cudaEventCreate(&D->link_ev1));
        }
        CSG_CUDA(cudaEventRecord(D->link_ev0, stream));
    }
    if (geometry == CSG_GEOM_MINKOWSKI_2D)
        link_kernel<GEOM_M2><<<(unsigned)ntiles, LK_THREADS, 0, stream>>>(coords, N, stride, rel_bits, nB);
    else if (geometry == CSG_GEOM_MINKOWSKI_4D)
        link_kernel<GEOM_M4><<<(unsigned)ntiles, LK_THREADS, 0, stream>>>(coords, N, stride, rel_bits, nB);
    else
        link_kernel<GEOM_DS2><<<(unsigned)ntiles, LK_THREADS, 0, stream>>>(coords, N, stride, rel_bits, nB);
    CSG_CUDA(cudaGetLastError());
    ++g.launches;
    if (g.timing) {
        CSG_CUDA(cudaEventRecord(D->link_ev1, stream));
        D->link_timed = true;
    }
    return CSG_OK;
}

// Library-owned device buffer of the host entry points; grows, never shrinks.  Growing frees the old buffer, which
// is safe here because those entry points synchronise their stream before they return.
static int ensure_buffer(void** ptr, size_t* have, size_t want) {
    if (*have >= want) return CSG_OK;
    if (*ptr) CSG_CUDA(cudaFree(*ptr));
    *ptr = nullptr;
    *have = 0;
    CSG_CUDA(cudaMalloc(ptr, want));
    *have = want;
    return CSG_OK;
}

static void release_device(Device* D) {
    for (TileList& t : D->tiles) cudaFree(t.d);
    for (ChunkTiles* c : D->chunk_tiles) {
        cudaFree(c->d);
        cudaFree(c->d_need);
        delete c;
    }
    if (D->d_bits) cudaFree(D->d_bits);
    if (D->d_counts) cudaFree(D->d_counts);
    if (D->d_S) cudaFree(D->d_S);
    if (D->d_coords) cudaFree(D->d_coords);
    if (D->d_progress) cudaFree(D->d_progress);
    if (D->d_landed) cudaFree(D->d_landed);
    for (uint32_t* p : D->d_occ) if (p) cudaFree(p);
    for (uint32_t* p : D->occ_retired) cudaFree(p);
    for (auto& kv : D->fused_ws) cudaFree(kv.second);
    for (cudaEvent_t e : D->chunk_ev) cudaEventDestroy(e);
    if (D->copy_stream) cudaStreamDestroy(D->copy_stream);
    if (D->occ_stream) cudaStreamDestroy(D->occ_stream);
    if (D->host_stream) cudaStreamDestroy(D->host_stream);
    if (D->link_ev0) cudaEventDestroy(D->link_ev0);
    if (D->link_ev1) cudaEventDestroy(D->link_ev1);
    for (int k = 0; k < TIMING_RING; ++k) {
        if (D->ev0[k]) cudaEventDestroy(D->ev0[k]);
        if (D->ev1[k]) cudaEventDestroy(D->ev1[k]);
    }
    delete D;
}

// ---------------------------------------------------------------------------------------------- csg_action_noalloc
// Scratch of the entry point that allocates nothing (include/csg.h): the workspace of the fused small-set launch
// (bitset_kernel.cuh: BitsetFusedWs = 1024 bins + the last-CTA ticket, 8200 bytes) in a file-scope device array instead of
// a cudaMalloc'ed buffer.  Every GPU that loads libcsg.so holds these 8448 bytes until the process exits.  In host
// code the NAME of the array is a host-side stand-in, not a device address: the kernel gets the address that
// cudaGetSymbolAddress returned for the device it runs on (noalloc_setup, once per device, with that device current).
constexpr size_t NOALLOC_SCRATCH_BYTES = 8448;
static_assert(sizeof(BitsetFusedWs) <= NOALLOC_SCRATCH_BYTES, "static scratch too small for the fused workspace");
static __device__ __align__(256) unsigned char csg_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

struct NoallocDevice {                  // plain static table: this path must not touch the heap-allocated Device state
    BitsetFusedWs* ws = nullptr;        // device address of csg_noalloc_scratch on this device
    int sm_count = 0;
};
static NoallocDevice g_noalloc[MAX_DEVICES];

// Set-up for the CURRENT device: device address of the scratch array and the SM count.  No allocation.
static int noalloc_setup(NoallocDevice** out) {
    int ord = 0;
    CSG_CUDA(cudaGetDevice(&ord));
    if (ord < 0 || ord >= MAX_DEVICES) {
        snprintf(g.cuda_msg, sizeof(g.cuda_msg), "device ordinal %d out of range", ord);
        return CSG_E_CUDA;
    }
    NoallocDevice& nd = g_noalloc[ord];
    if (!nd.ws) {
        int major = 0, sms = 0;
        CSG_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, ord));
        CSG_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ord));
        if (major != 10) {
            snprintf(g.cuda_msg, sizeof(g.cuda_msg), "device is sm_%dx; libcsg is built for sm_100a only", major);
            return CSG_E_CUDA;
        }
        void* ptr = nullptr;
        CSG_CUDA(cudaGetSymbolAddress(&ptr, csg_noalloc_scratch));
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255)) {
            snprintf(g.cuda_msg, sizeof(g.cuda_msg), "cudaGetSymbolAddress returned an unusable address for the static scratch");
            return CSG_E_CUDA;
        }
        nd.sm_count = sms;
        nd.ws = reinterpret_cast<BitsetFusedWs*>(ptr);
    }
    *out = &nd;
    return CSG_OK;
}

}  // namespace csg

using namespace csg;

extern "C" {

int64_t csg_row_stride_words(int64_t N) { return N < 1 ? 0 : 4 * ((N + 255) / 256); }

int csg_action(const uint64_t* rel_bits, int64_t N, int dim, double eps, int kmax, int64_t* counts, double* S,
               cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g.mu);
    int rc = validate(rel_bits, N, dim, eps, kmax, counts, S);
    if (rc) return rc;
    if ((reinterpret_cast<uintptr_t>(rel_bits) & 15) || (reinterpret_cast<uintptr_t>(counts) & 7) ||
        (reinterpret_cast<uintptr_t>(S) & 7))
        return CSG_E_ALIGN;
    Device* D = nullptr;
    if ((rc = current_device(&D))) return rc;
    return action_device(D, rel_bits, N, dim, eps, kmax, reinterpret_cast<long long*>(counts), S, stream);
}

int csg_action_partial(const uint64_t* rel_bits, int64_t N, int kmax, int shard, int nshards, int64_t* counts,
                       cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (!rel_bits || !counts) return CSG_E_NULL;
    if (N < 1 || N > CSG_MAX_N) return CSG_E_SIZE;
    if (kmax < 0 || kmax > CSG_MAX_KMAX) return CSG_E_KMAX;
    if (nshards < 1 || shard < 0 || shard >= nshards) return CSG_E_SHARD;
    if ((reinterpret_cast<uintptr_t>(rel_bits) & 15) || (reinterpret_cast<uintptr_t>(counts) & 7)) return CSG_E_ALIGN;
    Device* D = nullptr;
    int rc = current_device(&D);
    if (rc) return rc;
    return interval_device(D, rel_bits, N, kmax, shard, nshards, 0, reinterpret_cast<long long*>(counts), stream);
}

int csg_action_finish(const int64_t* counts, int64_t N, int dim, double eps, int kmax, double* S,
                      cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g.mu);
    int rc = validate(counts, N, dim, eps, kmax, counts, S);
    if (rc) return rc;
    if ((reinterpret_cast<uintptr_t>(counts) & 7) || (reinterpret_cast<uintptr_t>(S) & 7)) return CSG_E_ALIGN;
    Device* D = nullptr;
    if ((rc = current_device(&D))) return rc;
    return finish_device(reinterpret_cast<const long long*>(counts), N, dim, eps, kmax, S, stream);
}

int csg_action_batch(const uint64_t* rel_bits, int64_t N, int64_t batch, int dim, double eps, int kmax,
                     int64_t* counts, double* S, cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g.mu);
    int rc = validate(rel_bits, N, dim, eps, kmax, counts, S);
    if (rc) return rc;
    if (batch < 1 || batch > CSG_MAX_BATCH || batch * N >= (1LL << 31)) return CSG_E_SIZE;
    if ((reinterpret_cast<uintptr_t>(rel_bits) & 15) || (reinterpret_cast<uintptr_t>(counts) & 7) ||
        (reinterpret_cast<uintptr_t>(S) & 7))
        return CSG_E_ALIGN;
    Device* D = nullptr;
    if ((rc = current_device(&D))) return rc;
    const long long stride = csg_row_stride_words(N);
    const long long set_words = N * stride;
    long long* c = reinterpret_cast<long long*>(counts);
    const int variant = effective_batch_variant(N);
    if (variant == CSG_VARIANT_BITSET) {
        // one launch for the whole batch: grid.y = causal set, grid.x = CTAs per set sized so that the grid
        // still fills the machine (2 CTAs per SM) when the batch alone does not
        CSG_CUDA(cudaMemsetAsync(c, 0, (size_t)batch * (kmax + 1) * sizeof(long long), stream));
        const long long nb = (N + BS_T - 1) / BS_T;
        const long long ntiles = nb * (nb + 1) / 2;
        const long long per_set = std::max<long long>(1, (2LL * D->sm_count + batch - 1) / batch);
        const dim3 grid((unsigned)std::min<long long>(ntiles, per_set), (unsigned)batch);
        bitset_action_kernel<<<grid, BS_THREADS, 0, stream>>>(reinterpret_cast<const uint32_t*>(rel_bits), N, stride * 2,
                                                               kmax, reinterpret_cast<unsigned long long*>(c), nb, ntiles,
                                                               0, 1, set_words * 2, kmax + 1, nullptr, 0, 1.0, nullptr);
        CSG_CUDA(cudaGetLastError());
        ++g.launches;
    } else if (batch == 1 || N * stride * 8 > TILE_L2_BYTES) {
        // large sets fill the machine on their own (and take the patch schedule, the throttle and the block-sparse
        // sweep): one tensor launch per set, back to back on the stream
        for (int64_t b = 0; b < batch; ++b) {
            rc = interval_device(D, rel_bits + b * set_words, N, kmax, 0, 1, dim, c + b * (kmax + 1), stream);
            if (rc) return rc;
        }
    } else {
        // sets within L2: persistent tensor launches over the tiles of MANY sets at once, deepest first across the sets, so
        // that the machine is full whatever the size of a single set and there is no launch tail per set.  A launch
        // takes a power-of-two number of sets (64 sets: one launch; 100 sets: 64 + 32 + 4), so that the cached tile
        // lists are one per power of two and N -- not one per batch size a Monte-Carlo code happens to use -- and at
        // most BATCH_MAX_TILES entries each.
        const int kind = variant == CSG_VARIANT_TENSOR_FP4 ? KIND_FP4 : KIND_I8;
        const long long nB = (N + TC_T - 1) / TC_T, tiles_per_set = nB * (nB + 1) / 2;
        const long long max_group = std::max<long long>(1, BATCH_MAX_TILES / tiles_per_set);
        CSG_CUDA(cudaMemsetAsync(c, 0, (size_t)batch * (kmax + 1) * sizeof(long long), stream));
        for (int64_t b0 = 0; b0 < batch;) {
            long long nb = 1;
            while (2 * nb <= std::min<long long>(batch - b0, max_group)) nb *= 2;
            if (nb == 1) {          // a single set left over: the ordinary launch adds into its (zeroed) histogram
                const TileList* tl = nullptr;
                if ((rc = ensure_tiles(D, N, 0, 1, &tl))) return rc;
                rc = launch_tensor(D, kind, rel_bits + b0 * set_words, N, stride, kmax, c + b0 * (kmax + 1), tl->d, tl->n, nullptr,
                                   nullptr, nullptr, nullptr, stream);
            } else {
                const TileList* tl = nullptr;
                if ((rc = ensure_batch_tiles(D, N, (int)nb, &tl))) return rc;
                rc = launch_tensor(D, kind, rel_bits + b0 * set_words, N, stride, kmax, c + b0 * (kmax + 1), tl->d, tl->n, nullptr,
                                   nullptr, nullptr, nullptr, stream, (int)nb);
            }
            if (rc) return rc;
            b0 += nb;
        }
    }
    finish_action_kernel<<<(unsigned)batch, FIN_THREADS, 0, stream>>>(c, N, dim, eps, kmax, S);
    CSG_CUDA(cudaGetLastError());
    ++g.launches;
    return CSG_OK;
}

int64_t csg_tile_schedule(int64_t N, int shard, int nshards, int32_t* tiles_ij, int64_t capacity) {
    if (N < 1 || N > CSG_MAX_N) return CSG_E_SIZE;
    if (nshards < 1 || shard < 0 || shard >= nshards) return CSG_E_SHARD;
    std::vector<int2> tiles;
    build_tile_schedule(N, shard, nshards, tiles);
    if (tiles_ij)
        for (int64_t t = 0; t < (int64_t)tiles.size() && t < capacity; ++t) {
            tiles_ij[2 * t] = tiles[t].x;
            tiles_ij[2 * t + 1] = tiles[t].y;
        }
    return (int64_t)tiles.size();
}

int csg_action_host(const uint64_t* rel_bits_host, int64_t N, int dim, double eps, int kmax, int64_t* counts_host,
                    double* S_host) {
    std::lock_guard<std::mutex> lock(g.mu);
    int rc = validate(rel_bits_host, N, dim, eps, kmax, counts_host, S_host);
    if (rc) return rc;
    Device* D = nullptr;
    if ((rc = current_device(&D))) return rc;
    if (!D->host_stream) CSG_CUDA(cudaStreamCreateWithFlags(&D->host_stream, cudaStreamNonBlocking));
    const size_t bits_bytes = (size_t)N * (size_t)csg_row_stride_words(N) * sizeof(uint64_t);
    const size_t counts_bytes = (size_t)(kmax + 1) * sizeof(long long);
    if ((rc = ensure_buffer(reinterpret_cast<void**>(&D->d_bits), &D->d_bits_bytes, bits_bytes))) return rc;
    if ((rc = ensure_buffer(reinterpret_cast<void**>(&D->d_counts), &D->d_counts_bytes, counts_bytes))) return rc;
    if (!D->d_S) CSG_CUDA(cudaMalloc(&D->d_S, sizeof(double)));
    const int variant = effective_variant(N);
    if (variant != CSG_VARIANT_BITSET && bits_bytes >= (size_t)HOST_PIPELINE_MIN_BYTES) {
        rc = interval_host_pipelined(D, rel_bits_host, D->d_bits, N, kmax,
                                     variant == CSG_VARIANT_TENSOR_FP4 ? KIND_FP4 : KIND_I8, dim, D->d_counts, D->host_stream);
        if (rc) {
            cudaStreamSynchronize(D->host_stream);     // never leave a gated launch or a copy behind an error return
            cudaStreamSynchronize(D->copy_stream);
            if (D->occ_stream) cudaStreamSynchronize(D->occ_stream);
            return rc;
        }
        rc = finish_device(D->d_counts, N, dim, eps, kmax, D->d_S, D->host_stream);
    } else {
        CSG_CUDA(cudaMemcpyAsync(D->d_bits, rel_bits_host, bits_bytes, cudaMemcpyHostToDevice, D->host_stream));
        rc = action_device(D, D->d_bits, N, dim, eps, kmax, D->d_counts, D->d_S, D->host_stream);
    }
    if (rc) return rc;
    CSG_CUDA(cudaMemcpyAsync(counts_host, D->d_counts, counts_bytes, cudaMemcpyDeviceToHost, D->host_stream));
    CSG_CUDA(cudaMemcpyAsync(S_host, D->d_S, sizeof(double), cudaMemcpyDeviceToHost, D->host_stream));
    CSG_CUDA(cudaStreamSynchronize(D->host_stream));
    return CSG_OK;
}

int csg_link(const double* coords, int64_t N, int geometry, uint64_t* rel_bits, cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (!coords || !rel_bits) return CSG_E_NULL;
    if (N < 1 || N > CSG_MAX_N) return CSG_E_SIZE;
    if (geometry < CSG_GEOM_MINKOWSKI_2D || geometry > CSG_GEOM_DESITTER_2D) return CSG_E_GEOMETRY;
    if ((reinterpret_cast<uintptr_t>(rel_bits) & 15) || (reinterpret_cast<uintptr_t>(coords) & 7)) return CSG_E_ALIGN;
    Device* D = nullptr;
    int rc = current_device(&D);
    if (rc) return rc;
    return link_device(D, coords, N, geometry, rel_bits, stream);
}

int csg_causet_action_host(const double* coords_host, int64_t N, int geometry, double eps, int kmax,
                           int64_t* counts_host, double* S_host) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (geometry < CSG_GEOM_MINKOWSKI_2D || geometry > CSG_GEOM_DESITTER_2D) return CSG_E_GEOMETRY;
    const int dim = geometry_dim(geometry);
    int rc = validate(coords_host, N, dim, eps, kmax, counts_host, S_host);
    if (rc) return rc;
    Device* D = nullptr;
    if ((rc = current_device(&D))) return rc;
    if (!D->host_stream) CSG_CUDA(cudaStreamCreateWithFlags(&D->host_stream, cudaStreamNonBlocking));
    const size_t coords_bytes = (size_t)N * dim * sizeof(double);
    const size_t bits_bytes = (size_t)N * (size_t)csg_row_stride_words(N) * sizeof(uint64_t);
    const size_t counts_bytes = (size_t)(kmax + 1) * sizeof(long long);
    if ((rc = ensure_buffer(reinterpret_cast<void**>(&D->d_coords), &D->d_coords_bytes, coords_bytes))) return rc;
    if ((rc = ensure_buffer(reinterpret_cast<void**>(&D->d_bits), &D->d_bits_bytes, bits_bytes))) return rc;
    if ((rc = ensure_buffer(reinterpret_cast<void**>(&D->d_counts), &D->d_counts_bytes, counts_bytes))) return rc;
    if (!D->d_S) CSG_CUDA(cudaMalloc(&D->d_S, sizeof(double)));
    CSG_CUDA(cudaMemcpyAsync(D->d_coords, coords_host, coords_bytes, cudaMemcpyHostToDevice, D->host_stream));
    rc = link_device(D, D->d_coords, N, geometry, D->d_bits, D->host_stream);
    if (rc) return rc;
    rc = action_device(D, D->d_bits, N, dim, eps, kmax, D->d_counts, D->d_S, D->host_stream);
    if (rc) return rc;
    CSG_CUDA(cudaMemcpyAsync(counts_host, D->d_counts, counts_bytes, cudaMemcpyDeviceToHost, D->host_stream));
    CSG_CUDA(cudaMemcpyAsync(S_host, D->d_S, sizeof(double), cudaMemcpyDeviceToHost, D->host_stream));
    CSG_CUDA(cudaStreamSynchronize(D->host_stream));
    return CSG_OK;
}

int csg_last_link_ms(float* ms) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (!ms) return CSG_E_NULL;
    Device* D = nullptr;
    int rc = current_device(&D);
    if (rc) return rc;
    if (!D->link_timed) {
        snprintf(g.cuda_msg, sizeof(g.cuda_msg), "kernel timing: no timed csg_link call so far");
        return CSG_E_CUDA;
    }
    CSG_CUDA(cudaEventSynchronize(D->link_ev1));
    CSG_CUDA(cudaEventElapsedTime(ms, D->link_ev0, D->link_ev1));
    return CSG_OK;
}

int csg_interval_sizes(const uint64_t* rel_bits, int64_t N, const int64_t* pairs_ij, int64_t npairs, int32_t* n_out,
                       cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (!rel_bits || (npairs > 0 && (!pairs_ij || !n_out))) return CSG_E_NULL;
    if (N < 1 || N > CSG_MAX_N || npairs < 0) return CSG_E_SIZE;
    if (reinterpret_cast<uintptr_t>(rel_bits) & 15) return CSG_E_ALIGN;
    Device* D = nullptr;
    int rc = current_device(&D);
    if (rc) return rc;
    if (npairs == 0) return CSG_OK;
    const int warps_per_block = 8;
    const long long blocks = (npairs + warps_per_block - 1) / warps_per_block;
    pair_interval_kernel<<<(unsigned)blocks, warps_per_block * 32, 0, stream>>>(
        reinterpret_cast<const uint32_t*>(rel_bits), N, csg_row_stride_words(N) * 2,
        reinterpret_cast<const long long*>(pairs_ij), npairs, n_out);
    CSG_CUDA(cudaGetLastError());
    ++g.launches;
    return CSG_OK;
}

int csg_tile_interval_sizes(const uint64_t* rel_bits, int64_t N, const int32_t* tiles_ij_host, int64_t ntiles,
                            int32_t* n_out, cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (!rel_bits || (ntiles > 0 && (!tiles_ij_host || !n_out))) return CSG_E_NULL;
    if (N < 1 || N > CSG_MAX_N || ntiles < 0 || ntiles > (1 << 15)) return CSG_E_SIZE;
    if ((reinterpret_cast<uintptr_t>(rel_bits) & 15) || (reinterpret_cast<uintptr_t>(n_out) & 3)) return CSG_E_ALIGN;
    const int nB = (int)((N + TC_T - 1) / TC_T);
    for (int64_t t = 0; t < ntiles; ++t)
        if (tiles_ij_host[2 * t] < 0 || tiles_ij_host[2 * t] > tiles_ij_host[2 * t + 1] || tiles_ij_host[2 * t + 1] >= nB)
            return CSG_E_SIZE;
    const int variant = effective_variant(N);
    if (variant == CSG_VARIANT_BITSET) return CSG_E_UNSUPPORTED;
    Device* D = nullptr;
    int rc = current_device(&D);
    if (rc) return rc;
    if (ntiles == 0) return CSG_OK;
    // a test hook: temporary tile list, synchronous
    int2* d_tiles = nullptr;
    CSG_CUDA(cudaMalloc(&d_tiles, (size_t)ntiles * sizeof(int2)));
    cudaError_t e = cudaMemcpy(d_tiles, tiles_ij_host, (size_t)ntiles * sizeof(int2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        const int kind = variant == CSG_VARIANT_TENSOR_FP4 ? KIND_FP4 : KIND_I8;
        const uint32_t* occ = nullptr;
        rc = occupancy_pass(D, kind, rel_bits, N, csg_row_stride_words(N), 0, &occ, stream);
        if (rc == CSG_OK)
            rc = launch_tensor(D, kind, rel_bits, N, csg_row_stride_words(N), 0, nullptr, d_tiles, (int)ntiles, nullptr, nullptr,
                               n_out, occ, stream);
        e = cudaStreamSynchronize(stream);
    }
    cudaFree(d_tiles);
    if (e != cudaSuccess) return cuda_fail(e, "csg_tile_interval_sizes");
    return rc;
}

int csg_noalloc_setup(void) {
    std::lock_guard<std::mutex> lock(g.mu);
    NoallocDevice* nd = nullptr;
    return noalloc_setup(&nd);
}

int csg_action_noalloc(const uint64_t* rel_bits, int64_t N, int dim, double eps, int kmax, int64_t* counts, double* S,
                       cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g.mu);
    int rc = validate(rel_bits, N, dim, eps, kmax, counts, S);
    if (rc) return rc;
    if (N > CSG_NOALLOC_MAX_N || kmax > CSG_NOALLOC_MAX_KMAX) return CSG_E_NOALLOC_LIMIT;
    if ((reinterpret_cast<uintptr_t>(rel_bits) & 15) || (reinterpret_cast<uintptr_t>(counts) & 7) ||
        (reinterpret_cast<uintptr_t>(S) & 7))
        return CSG_E_ALIGN;
    NoallocDevice* nd = nullptr;
    if ((rc = noalloc_setup(&nd))) return rc;          // a lookup after the first call on this device
    // Every call shares the scratch and it keeps what the last call left there (zeros after a completed launch, anything
    // after a failed or aborted one): clear the bins and the ticket on the caller's stream first.
    CSG_CUDA(cudaMemsetAsync(nd->ws, 0, sizeof(BitsetFusedWs), stream));
    const long long stride = csg_row_stride_words(N);
    const long long nb = (N + BS_T - 1) / BS_T;
    const long long ntiles = nb * (nb + 1) / 2;
    const int grid = (int)std::max<long long>(1, std::min<long long>(ntiles, (long long)nd->sm_count * 2));
    bitset_action_kernel<<<grid, BS_THREADS, 0, stream>>>(reinterpret_cast<const uint32_t*>(rel_bits), N, stride * 2, kmax,
                                                           reinterpret_cast<unsigned long long*>(counts), nb, ntiles, 0, 1, 0,
                                                           0, nd->ws, dim, eps, S);
    CSG_CUDA(cudaGetLastError());
    ++g.launches;
    return CSG_OK;
}

int csg_set_variant(int variant) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (variant < CSG_VARIANT_AUTO || variant > CSG_VARIANT_TENSOR_FP4)
        return CSG_E_VARIANT;
    g.variant = variant;
    return CSG_OK;
}

int csg_effective_variant(int64_t N) {
    std::lock_guard<std::mutex> lock(g.mu);
    return effective_variant(N);
}

int csg_set_throttle(int mode) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (mode < CSG_THROTTLE_AUTO || mode > CSG_THROTTLE_OFF) return CSG_E_VARIANT;
    g.throttle = mode;
    return CSG_OK;
}

int csg_set_sparse(int mode) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (mode < CSG_SPARSE_AUTO || mode > CSG_SPARSE_OFF) return CSG_E_VARIANT;
    g.sparse = mode;
    return CSG_OK;
}

int csg_set_host_pipeline(int mode) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (mode < CSG_HOST_PIPELINE_AUTO || mode > CSG_HOST_PIPELINE_CHUNKED) return CSG_E_VARIANT;
    g.host_pipeline = mode;
    return CSG_OK;
}

int64_t csg_occupancy_stride_words(int64_t N) { return N < 1 ? 0 : occ_stride_words(N); }

int csg_block_occupancy(const uint64_t* rel_bits, int64_t N, uint32_t* occ, cudaStream_t stream) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (!rel_bits || !occ) return CSG_E_NULL;
    if (N < 1 || N > CSG_MAX_N) return CSG_E_SIZE;
    if ((reinterpret_cast<uintptr_t>(rel_bits) & 15) || (reinterpret_cast<uintptr_t>(occ) & 3)) return CSG_E_ALIGN;
    Device* D = nullptr;
    int rc = current_device(&D);
    if (rc) return rc;
    const int nB = (int)((N + TC_T - 1) / TC_T), ostride = occ_stride_words(N);
    occupancy_kernel<<<dim3(ostride / OCC_WORDS_PER_CTA, nB), OCC_THREADS, 0, stream>>>(rel_bits, N, csg_row_stride_words(N), occ, ostride, 0);
    CSG_CUDA(cudaGetLastError());
    ++g.launches;
    return CSG_OK;
}

#ifdef CSG_ABLATE
int csg_set_debug(int bits) {
    std::lock_guard<std::mutex> lock(g.mu);
    g.debug = bits;
    return CSG_OK;
}
#endif

int csg_set_kernel_timing(int enable) {
    std::lock_guard<std::mutex> lock(g.mu);
    g.timing = enable != 0;
    if (!g.timing)
        for (Device* D : g.dev)
            if (D) D->timed_calls = 0;
    return CSG_OK;
}

static int kernel_ms_history(float* ms, int n) {
    if (!ms) return CSG_E_NULL;
    if (n < 1 || n > TIMING_RING) return CSG_E_SIZE;
    Device* D = nullptr;
    int rc = current_device(&D);
    if (rc) return rc;
    if (D->timed_calls < n) {
        snprintf(g.cuda_msg, sizeof(g.cuda_msg), "kernel timing: only %lld timed csg_action calls so far, %d asked",
                 D->timed_calls, n);
        return CSG_E_CUDA;
    }
    for (int k = 0; k < n; ++k) {
        const int slot = (int)((D->timed_calls - n + k) % TIMING_RING);
        CSG_CUDA(cudaEventSynchronize(D->ev1[slot]));
        CSG_CUDA(cudaEventElapsedTime(&ms[k], D->ev0[slot], D->ev1[slot]));
    }
    return CSG_OK;
}

int csg_last_kernel_ms(float* ms) {
    std::lock_guard<std::mutex> lock(g.mu);
    return kernel_ms_history(ms, 1);
}

int csg_kernel_ms_history(float* ms, int n) {
    std::lock_guard<std::mutex> lock(g.mu);
    return kernel_ms_history(ms, n);
}

int64_t csg_launch_count(void) {
    std::lock_guard<std::mutex> lock(g.mu);
    return g.launches;
}

int csg_measure_peak(int what, int iters, float* ms, double* units) {
    std::lock_guard<std::mutex> lock(g.mu);
    if (!ms || !units) return CSG_E_NULL;
    if (iters < 1 || what < CSG_PEAK_MMA_MXF4 || what > CSG_PEAK_ALU_LOP3) return CSG_E_SIZE;
    Device* D = nullptr;
    int rc = current_device(&D);
    if (rc) return rc;
    if ((rc = ensure_tensor_ready(D))) return rc;
    cudaEvent_t e0, e1;
    CSG_CUDA(cudaEventCreate(&e0));
    CSG_CUDA(cudaEventCreate(&e1));
    unsigned int* sink = nullptr;
    CSG_CUDA(cudaMalloc(&sink, sizeof(unsigned int)));
    const int clusters = D->sm_count / 2;
    cudaEventRecord(e0, 0);
    if (what == CSG_PEAK_MMA_MXF4) {
        tensor_peak_kernel<KIND_FP4><<<2 * clusters, TC_THREADS, TcTraits<KIND_FP4>::SMEM_BYTES>>>(iters, sink);
        *units = (double)clusters * iters * 4.0 * 256.0 * 256.0 * 64.0;          // MACs
    } else if (what == CSG_PEAK_MMA_I8) {
        tensor_peak_kernel<KIND_I8><<<2 * clusters, TC_THREADS, TcTraits<KIND_I8>::SMEM_BYTES>>>(iters, sink);
        *units = (double)clusters * iters * 4.0 * 256.0 * 256.0 * 32.0;
    } else {
        const int grid = D->sm_count * 8;
        if (what == CSG_PEAK_ALU_MIX) alu_peak_kernel<0><<<grid, ALU_PEAK_THREADS>>>(iters, sink);
        else if (what == CSG_PEAK_ALU_POPC) alu_peak_kernel<1><<<grid, ALU_PEAK_THREADS>>>(iters, sink);
        else alu_peak_kernel<2><<<grid, ALU_PEAK_THREADS>>>(iters, sink);
        *units = (double)grid * ALU_PEAK_THREADS * iters * 8.0;                   // lane-steps (MIX: 1 AND + 1 POPC + 1 ADD each)
    }
    cudaError_t e = cudaGetLastError();
    cudaEventRecord(e1, 0);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    ++g.launches;
    if (e != cudaSuccess) return cuda_fail(e, "csg_measure_peak");
    return CSG_OK;
}

const char* csg_strerror(int code) {
    switch (code) {
        case CSG_OK: return "success";
        case CSG_E_NULL: return "null pointer";
        case CSG_E_SIZE: return "N, npairs, ntiles or a tile index out of range";
        case CSG_E_ALIGN: return "misaligned buffer (rel_bits needs 16 bytes, counts and S 8 bytes)";
        case CSG_E_DIM: return "dim must be 2 or 4";
        case CSG_E_EPS: return "eps must be in (0, 1]";
        case CSG_E_KMAX: return "kmax out of range (local action needs kmax >= 2 in 2D, >= 3 in 4D)";
        case CSG_E_UNSUPPORTED: return "unsupported combination of arguments";
        case CSG_E_CUDA: return g.cuda_msg;
        case CSG_E_VARIANT: return "unknown variant or mode";
        case CSG_E_GEOMETRY: return "geometry must be CSG_GEOM_MINKOWSKI_2D, _MINKOWSKI_4D or _DESITTER_2D";
        case CSG_E_SHARD: return "shard must satisfy 0 <= shard < nshards";
        case CSG_E_NOALLOC_LIMIT:
            return "csg_action_noalloc: N > CSG_NOALLOC_MAX_N (4096) or kmax > CSG_NOALLOC_MAX_KMAX (1023): beyond its static scratch; use csg_action";
        default: return "unknown error code";
    }
}

int csg_shutdown(void) {
    std::lock_guard<std::mutex> lock(g.mu);
    for (int d = 0; d < MAX_DEVICES; ++d)
        if (g.dev[d]) {
            release_device(g.dev[d]);
            g.dev[d] = nullptr;
        }
    cudaGetLastError();
    return CSG_OK;
}

}  // extern "C"
