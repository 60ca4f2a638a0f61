"""paper_1709_03013_b200 -- thin Python binding of libcsg (include/csg.h).

Argument marshalling only: every step of the hot path (interval sizes, histogram, action) runs in the
hand-written sm_100a kernels behind the C ABI.  PyTorch is used for device memory and streams.
There is no CPU fallback: if libcsg.so is missing, importing the compute entry points fails loudly.

Functions carry the C names: csg_action, csg_action_host, csg_interval_sizes, csg_row_stride_words,
csg_set_variant, csg_effective_variant, csg_set_kernel_timing, csg_last_kernel_ms, csg_kernel_ms_history,
csg_launch_count, csg_action_partial, csg_action_finish, csg_tile_schedule, csg_link, csg_causet_action_host,
csg_last_link_ms, csg_action_batch, csg_tile_interval_sizes, csg_set_throttle, csg_set_sparse, csg_set_host_pipeline,
csg_occupancy_stride_words, csg_block_occupancy, csg_measure_peak, csg_noalloc_setup, csg_action_noalloc,
csg_strerror, csg_shutdown.
"""
import ctypes
import os

import numpy as np

from . import _build

VARIANT_AUTO, VARIANT_BITSET, VARIANT_TENSOR, VARIANT_TENSOR_FP4 = 0, 1, 2, 3
GEOM_MINKOWSKI_2D, GEOM_MINKOWSKI_4D, GEOM_DESITTER_2D = 0, 1, 2
THROTTLE_AUTO, THROTTLE_ON, THROTTLE_OFF = 0, 1, 2
SPARSE_AUTO, SPARSE_ON, SPARSE_OFF = 0, 1, 2
HOST_PIPELINE_AUTO, HOST_PIPELINE_CHUNKED = 0, 1
PEAK_MMA_MXF4, PEAK_MMA_I8, PEAK_ALU_MIX, PEAK_ALU_POPC, PEAK_ALU_LOP3 = 0, 1, 2, 3, 4
LIB_PATH = _build.LIB_PATH

EXPORTS = [
    "csg_row_stride_words", "csg_action", "csg_action_host", "csg_interval_sizes", "csg_set_variant",
    "csg_effective_variant", "csg_set_kernel_timing", "csg_last_kernel_ms", "csg_kernel_ms_history",
    "csg_launch_count", "csg_action_partial", "csg_action_finish", "csg_tile_schedule", "csg_link",
    "csg_causet_action_host", "csg_last_link_ms", "csg_action_batch", "csg_tile_interval_sizes", "csg_set_throttle",
    "csg_measure_peak", "csg_set_sparse", "csg_occupancy_stride_words", "csg_block_occupancy",
    "csg_set_host_pipeline", "csg_noalloc_setup", "csg_action_noalloc",
    "csg_strerror", "csg_shutdown",
]

_lib = None


class CsgError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("libcsg error %d: %s" % (code, text))
        self.code = code


def build(force=False, verbose=False):
    """Compile libcsg.so in-tree (nvcc, sm_100a)."""
    return _build.build(force=force, verbose=verbose)


def load():
    """dlopen libcsg.so and declare the prototypes of include/csg.h.  Raises if the library is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, ci, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
    lib.csg_row_stride_words.argtypes = [i64]
    lib.csg_row_stride_words.restype = i64
    lib.csg_action.argtypes = [vp, i64, ci, dbl, ci, vp, vp, vp]
    lib.csg_action.restype = ci
    lib.csg_action_host.argtypes = [vp, i64, ci, dbl, ci, vp, vp]
    lib.csg_action_host.restype = ci
    lib.csg_action_partial.argtypes = [vp, i64, ci, ci, ci, vp, vp]
    lib.csg_action_partial.restype = ci
    lib.csg_action_finish.argtypes = [vp, i64, ci, dbl, ci, vp, vp]
    lib.csg_action_finish.restype = ci
    lib.csg_tile_schedule.argtypes = [i64, ci, ci, vp, i64]
    lib.csg_tile_schedule.restype = i64
    lib.csg_action_batch.argtypes = [vp, i64, i64, ci, dbl, ci, vp, vp, vp]
    lib.csg_action_batch.restype = ci
    lib.csg_link.argtypes = [vp, i64, ci, vp, vp]
    lib.csg_link.restype = ci
    lib.csg_causet_action_host.argtypes = [vp, i64, ci, dbl, ci, vp, vp]
    lib.csg_causet_action_host.restype = ci
    lib.csg_last_link_ms.argtypes = [ctypes.POINTER(ctypes.c_float)]
    lib.csg_last_link_ms.restype = ci
    lib.csg_interval_sizes.argtypes = [vp, i64, vp, i64, vp, vp]
    lib.csg_interval_sizes.restype = ci
    lib.csg_tile_interval_sizes.argtypes = [vp, i64, vp, i64, vp, vp]
    lib.csg_tile_interval_sizes.restype = ci
    lib.csg_set_throttle.argtypes = [ci]
    lib.csg_set_throttle.restype = ci
    lib.csg_set_sparse.argtypes = [ci]
    lib.csg_set_sparse.restype = ci
    lib.csg_noalloc_setup.argtypes = []
    lib.csg_noalloc_setup.restype = ci
    lib.csg_action_noalloc.argtypes = [vp, i64, ci, dbl, ci, vp, vp, vp]
    lib.csg_action_noalloc.restype = ci
    lib.csg_set_host_pipeline.argtypes = [ci]
    lib.csg_set_host_pipeline.restype = ci
    lib.csg_occupancy_stride_words.argtypes = [i64]
    lib.csg_occupancy_stride_words.restype = i64
    lib.csg_block_occupancy.argtypes = [vp, i64, vp, vp]
    lib.csg_block_occupancy.restype = ci
    lib.csg_measure_peak.argtypes = [ci, ci, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_double)]
    lib.csg_measure_peak.restype = ci
    lib.csg_set_variant.argtypes = [ci]
    lib.csg_set_variant.restype = ci
    lib.csg_effective_variant.argtypes = [i64]
    lib.csg_effective_variant.restype = ci
    lib.csg_set_kernel_timing.argtypes = [ci]
    lib.csg_set_kernel_timing.restype = ci
    lib.csg_last_kernel_ms.argtypes = [ctypes.POINTER(ctypes.c_float)]
    lib.csg_last_kernel_ms.restype = ci
    lib.csg_kernel_ms_history.argtypes = [ctypes.POINTER(ctypes.c_float), ci]
    lib.csg_kernel_ms_history.restype = ci
    lib.csg_launch_count.argtypes = []
    lib.csg_launch_count.restype = i64
    lib.csg_strerror.argtypes = [ci]
    lib.csg_strerror.restype = ctypes.c_char_p
    lib.csg_shutdown.argtypes = []
    lib.csg_shutdown.restype = ci
    _lib = lib
    return lib


def _check(code):
    if code != 0:
        raise CsgError(code, csg_strerror(code))


def csg_strerror(code):
    return load().csg_strerror(int(code)).decode()


def csg_row_stride_words(N):
    return int(load().csg_row_stride_words(int(N)))


def _stream_handle(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def to_device(bits, device="cuda"):
    """numpy (N, stride) uint64 relation matrix -> CUDA int64 tensor holding the same words."""
    import torch
    b = np.ascontiguousarray(bits, dtype=np.uint64)
    return torch.from_numpy(b.view(np.int64)).to(device)


def csg_action(rel_bits, N, dim, eps, kmax, counts=None, S=None, stream=None):
    """int csg_action(rel_bits, N, dim, eps, kmax, counts, S, stream) -- see include/csg.h.

    rel_bits: CUDA tensor of 64-bit words, N rows of csg_row_stride_words(N).  counts (int64, kmax+1) and
    S (float64, 1) are allocated on the same device when not given.  Returns (counts, S) device tensors;
    nothing is synchronised."""
    import torch
    lib = load()
    assert rel_bits.is_cuda and rel_bits.element_size() == 8 and rel_bits.is_contiguous()
    assert rel_bits.numel() >= int(N) * csg_row_stride_words(N)
    if counts is None:
        counts = torch.empty(max(int(kmax), 0) + 1, dtype=torch.int64, device=rel_bits.device)
    if S is None:
        S = torch.empty(1, dtype=torch.float64, device=rel_bits.device)
    _check(lib.csg_action(rel_bits.data_ptr(), int(N), int(dim), float(eps), int(kmax), counts.data_ptr(),
                          S.data_ptr(), _stream_handle(stream)))
    return counts, S


NOALLOC_MAX_N, NOALLOC_MAX_KMAX = 4096, 1023


def csg_noalloc_setup():
    _check(load().csg_noalloc_setup())


def csg_action_noalloc(rel_bits, N, dim, eps, kmax, counts, S, stream=None):
    """int csg_action_noalloc(rel_bits, N, dim, eps, kmax, counts, S, stream): csg_action for small sets with its scratch
    in a static device array (include/csg.h).  The caller passes every buffer (device tensors): nothing is allocated
    here either.  Returns (counts, S); nothing is synchronised."""
    lib = load()
    assert rel_bits.is_cuda and rel_bits.element_size() == 8 and rel_bits.is_contiguous()
    assert counts.is_cuda and counts.element_size() == 8 and S.is_cuda and S.element_size() == 8
    _check(lib.csg_action_noalloc(rel_bits.data_ptr(), int(N), int(dim), float(eps), int(kmax), counts.data_ptr(),
                                  S.data_ptr(), _stream_handle(stream)))
    return counts, S


def csg_action_batch(rel_bits, N, batch, dim, eps, kmax, counts=None, S=None, stream=None):
    """int csg_action_batch(rel_bits, N, batch, dim, eps, kmax, counts, S, stream): `batch` causal sets of N elements,
    matrices back to back in one CUDA tensor.  Returns (counts (batch, kmax+1) int64, S (batch,) float64)."""
    import torch
    lib = load()
    assert rel_bits.is_cuda and rel_bits.element_size() == 8 and rel_bits.is_contiguous()
    assert rel_bits.numel() >= int(batch) * int(N) * csg_row_stride_words(N)
    if counts is None:
        counts = torch.empty((int(batch), max(int(kmax), 0) + 1), dtype=torch.int64, device=rel_bits.device)
    if S is None:
        S = torch.empty(int(batch), dtype=torch.float64, device=rel_bits.device)
    _check(lib.csg_action_batch(rel_bits.data_ptr(), int(N), int(batch), int(dim), float(eps), int(kmax),
                                counts.data_ptr(), S.data_ptr(), _stream_handle(stream)))
    return counts, S


def csg_action_partial(rel_bits, N, kmax, shard, nshards, counts=None, stream=None):
    """int csg_action_partial(rel_bits, N, kmax, shard, nshards, counts, stream): abundances of one shard of the
    pair tiles (device tensors; nothing is synchronised).  Returns counts."""
    import torch
    lib = load()
    assert rel_bits.is_cuda and rel_bits.element_size() == 8 and rel_bits.is_contiguous()
    assert rel_bits.numel() >= int(N) * csg_row_stride_words(N)
    if counts is None:
        counts = torch.empty(max(int(kmax), 0) + 1, dtype=torch.int64, device=rel_bits.device)
    _check(lib.csg_action_partial(rel_bits.data_ptr(), int(N), int(kmax), int(shard), int(nshards), counts.data_ptr(),
                                  _stream_handle(stream)))
    return counts


def csg_action_finish(counts, N, dim, eps, kmax, S=None, stream=None):
    """int csg_action_finish(counts, N, dim, eps, kmax, S, stream): summed abundances -> action.  Returns S."""
    import torch
    lib = load()
    assert counts.is_cuda and counts.dtype == torch.int64 and counts.numel() >= int(kmax) + 1
    if S is None:
        S = torch.empty(1, dtype=torch.float64, device=counts.device)
    _check(lib.csg_action_finish(counts.data_ptr(), int(N), int(dim), float(eps), int(kmax), S.data_ptr(),
                                 _stream_handle(stream)))
    return S


def csg_tile_schedule(N, shard=0, nshards=1):
    """int64 csg_tile_schedule(N, shard, nshards, tiles_ij, capacity): host logic, needs no device.
    Returns an (ntiles, 2) int32 numpy array of (I, J) block pairs in launch order."""
    lib = load()
    n = int(lib.csg_tile_schedule(int(N), int(shard), int(nshards), None, 0))
    if n < 0:
        _check(n)
    out = np.empty((n, 2), dtype=np.int32)
    if n:
        got = int(lib.csg_tile_schedule(int(N), int(shard), int(nshards), out.ctypes.data, n))
        assert got == n
    return out


def geometry_dim(geometry):
    return 4 if int(geometry) == GEOM_MINKOWSKI_4D else 2


def csg_link(coords, N, geometry, rel_bits=None, stream=None):
    """int csg_link(coords, N, geometry, rel_bits, stream): time-sorted coordinates (CUDA float64 tensor, N x dim)
    -> packed symmetric relation matrix (CUDA int64 tensor, N x csg_row_stride_words(N)).  Returns rel_bits."""
    import torch
    lib = load()
    assert coords.is_cuda and coords.dtype == torch.float64 and coords.is_contiguous()
    assert coords.numel() >= int(N) * geometry_dim(geometry)
    if rel_bits is None:
        rel_bits = torch.empty((int(N), csg_row_stride_words(N)), dtype=torch.int64, device=coords.device)
    assert rel_bits.is_cuda and rel_bits.element_size() == 8 and rel_bits.is_contiguous()
    assert rel_bits.numel() >= int(N) * csg_row_stride_words(N)
    _check(lib.csg_link(coords.data_ptr(), int(N), int(geometry), rel_bits.data_ptr(), _stream_handle(stream)))
    return rel_bits


def csg_causet_action_host(coords, N, geometry, eps, kmax):
    """int csg_causet_action_host(...) with HOST buffers: coords is a numpy float64 (N, dim) array or a (pinned)
    CPU torch tensor.  Returns (counts numpy int64[kmax+1], S float)."""
    lib = load()
    if isinstance(coords, np.ndarray):
        assert coords.dtype == np.float64 and coords.flags["C_CONTIGUOUS"]
        ptr, n = coords.ctypes.data, coords.size
    else:
        assert not coords.is_cuda and coords.element_size() == 8 and coords.is_contiguous()
        ptr, n = coords.data_ptr(), coords.numel()
    assert n >= int(N) * geometry_dim(geometry)
    counts = np.empty(max(int(kmax), 0) + 1, dtype=np.int64)
    S = np.empty(1, dtype=np.float64)
    _check(lib.csg_causet_action_host(ptr, int(N), int(geometry), float(eps), int(kmax), counts.ctypes.data,
                                      S.ctypes.data))
    return counts, float(S[0])


def csg_last_link_ms():
    ms = ctypes.c_float(0.0)
    _check(load().csg_last_link_ms(ctypes.byref(ms)))
    return float(ms.value)


def csg_action_host(rel_bits, N, dim, eps, kmax):
    """int csg_action_host(...) with HOST buffers: rel_bits is a numpy uint64 array or a (pinned) CPU torch
    tensor of 64-bit words.  Returns (counts numpy int64[kmax+1], S float)."""
    lib = load()
    if isinstance(rel_bits, np.ndarray):
        assert rel_bits.dtype in (np.uint64, np.int64) and rel_bits.flags["C_CONTIGUOUS"]
        ptr, nwords = rel_bits.ctypes.data, rel_bits.size
    else:
        assert not rel_bits.is_cuda and rel_bits.element_size() == 8 and rel_bits.is_contiguous()
        ptr, nwords = rel_bits.data_ptr(), rel_bits.numel()
    assert nwords >= int(N) * csg_row_stride_words(N)
    counts = np.empty(max(int(kmax), 0) + 1, dtype=np.int64)
    S = np.empty(1, dtype=np.float64)
    _check(lib.csg_action_host(ptr, int(N), int(dim), float(eps), int(kmax), counts.ctypes.data, S.ctypes.data))
    return counts, float(S[0])


def csg_interval_sizes(rel_bits, N, pairs_ij, n_out=None, stream=None):
    """Test hook: n_ij for listed pairs.  pairs_ij: CUDA int64 tensor (npairs, 2).  Returns int32 tensor."""
    import torch
    lib = load()
    assert rel_bits.is_cuda and pairs_ij.is_cuda and pairs_ij.dtype == torch.int64 and pairs_ij.is_contiguous()
    npairs = pairs_ij.numel() // 2
    if n_out is None:
        n_out = torch.empty(npairs, dtype=torch.int32, device=rel_bits.device)
    _check(lib.csg_interval_sizes(rel_bits.data_ptr(), int(N), pairs_ij.data_ptr(), npairs, n_out.data_ptr(),
                                  _stream_handle(stream)))
    return n_out


def csg_tile_interval_sizes(rel_bits, N, tiles_ij, n_out=None, stream=None):
    """Test hook: all n_ij of the listed 256 x 256 tiles from the tensor kernel itself.  tiles_ij: (ntiles, 2) int
    array-like of block pairs I <= J.  Returns a CUDA int32 tensor (ntiles, 256, 256), -1 where (i, j) is no related
    pair; synchronised."""
    import torch
    lib = load()
    tiles = np.ascontiguousarray(np.asarray(tiles_ij, dtype=np.int32).reshape(-1, 2))
    assert rel_bits.is_cuda and rel_bits.element_size() == 8 and rel_bits.is_contiguous()
    if n_out is None:
        n_out = torch.empty((tiles.shape[0], 256, 256), dtype=torch.int32, device=rel_bits.device)
    assert n_out.is_cuda and n_out.dtype == torch.int32 and n_out.numel() >= tiles.shape[0] * 65536
    _check(lib.csg_tile_interval_sizes(rel_bits.data_ptr(), int(N), tiles.ctypes.data, tiles.shape[0], n_out.data_ptr(),
                                       _stream_handle(stream)))
    return n_out


def csg_set_throttle(mode):
    _check(load().csg_set_throttle(int(mode)))


def csg_set_sparse(mode):
    _check(load().csg_set_sparse(int(mode)))


def csg_set_host_pipeline(mode):
    _check(load().csg_set_host_pipeline(int(mode)))


def csg_occupancy_stride_words(N):
    return int(load().csg_occupancy_stride_words(int(N)))


def csg_block_occupancy(rel_bits, N, occ=None, stream=None):
    """int csg_block_occupancy(rel_bits, N, occ, stream): occ = int32 CUDA tensor (ceil(N/256), stride) of bit words."""
    import torch
    assert rel_bits.is_cuda and rel_bits.element_size() == 8 and rel_bits.is_contiguous()
    if occ is None:
        occ = torch.empty(((int(N) + 255) // 256, csg_occupancy_stride_words(N)), dtype=torch.int32, device=rel_bits.device)
    assert occ.is_cuda and occ.dtype == torch.int32 and occ.is_contiguous()
    _check(load().csg_block_occupancy(rel_bits.data_ptr(), int(N), occ.data_ptr(), _stream_handle(stream)))
    return occ


def csg_measure_peak(what, iters):
    """int csg_measure_peak(what, iters, ms, units): returns (ms, units) of one bare peak kernel (PEAK_* ids)."""
    ms, units = ctypes.c_float(0.0), ctypes.c_double(0.0)
    _check(load().csg_measure_peak(int(what), int(iters), ctypes.byref(ms), ctypes.byref(units)))
    return float(ms.value), float(units.value)


def csg_set_variant(variant):
    _check(load().csg_set_variant(int(variant)))


def csg_effective_variant(N):
    return int(load().csg_effective_variant(int(N)))


def csg_set_kernel_timing(enable):
    _check(load().csg_set_kernel_timing(1 if enable else 0))


def csg_last_kernel_ms():
    ms = ctypes.c_float(0.0)
    _check(load().csg_last_kernel_ms(ctypes.byref(ms)))
    return float(ms.value)


def csg_kernel_ms_history(n):
    buf = (ctypes.c_float * int(n))()
    _check(load().csg_kernel_ms_history(buf, int(n)))
    return [float(x) for x in buf]


def csg_launch_count():
    return int(load().csg_launch_count())


def csg_shutdown():
    _check(load().csg_shutdown())
