"""ctypes front end of the C oracle (oracle/csg_oracle.c, oracle/alg5_packed.c).

Test infrastructure only (see oracle/__init__.py).  Every function cites the PAPER.md passage its C body
follows; the arithmetic lives in the C files, this module only marshals numpy arrays.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_SRCS = [os.path.join(_HERE, "csg_oracle.c"), os.path.join(_HERE, "alg5_packed.c"),
         os.path.join(_HERE, "link_oracle.c"), os.path.join(_HERE, "dominance2d.c")]
_lib = None

_i64 = ctypes.c_int64
_p_u64 = np.ctypeslib.ndpointer(dtype=np.uint64, flags="C_CONTIGUOUS")
_p_u8 = np.ctypeslib.ndpointer(dtype=np.uint8, flags="C_CONTIGUOUS")
_p_i64 = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def build(force=False):
    """Compile the oracle with gcc (plain -O2; OpenMP only drives the pair loops of Algorithm 5 and of the
    coordinate route; -mpopcnt because Algorithm 5's bit count IS the popcnt instruction, Alg. 3 --
    without it gcc calls a table routine and the restated algorithm runs 2.5x slower than the paper's own)."""
    newest = max(os.path.getmtime(s) for s in _SRCS)
    if not force and os.path.exists(_LIB_PATH) and os.path.getmtime(_LIB_PATH) >= newest:
        return _LIB_PATH
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-mpopcnt", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB_PATH] + _SRCS + ["-lm"]
    subprocess.run(cmd, check=True)
    return _LIB_PATH


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = ctypes.CDLL(_LIB_PATH)
    lib.csg_oracle_expand.argtypes = [_p_u64, _i64, _i64, _p_u8]
    lib.csg_oracle_expand.restype = None
    lib.csg_oracle_counts.argtypes = [_p_u8, _i64, _i64, _p_i64]
    lib.csg_oracle_counts.restype = None
    lib.csg_oracle_pair.argtypes = [_p_u64, _i64, _i64, _i64, _i64]
    lib.csg_oracle_pair.restype = _i64
    lib.csg_oracle_action_local.argtypes = [ctypes.c_int, _i64, _p_i64]
    lib.csg_oracle_action_local.restype = ctypes.c_double
    lib.csg_oracle_f2.argtypes = [_i64, ctypes.c_double]
    lib.csg_oracle_f2.restype = ctypes.c_double
    lib.csg_oracle_action_smeared_2d.argtypes = [_i64, _i64, _p_i64, ctypes.c_double,
                                                 ctypes.POINTER(ctypes.c_double)]
    lib.csg_oracle_action_smeared_2d.restype = ctypes.c_double
    lib.csg_oracle_f4.argtypes = [_i64, ctypes.c_double]
    lib.csg_oracle_f4.restype = ctypes.c_double
    lib.csg_oracle_action_smeared_4d.argtypes = [_i64, _i64, _p_i64, ctypes.c_double,
                                                 ctypes.POINTER(ctypes.c_double)]
    lib.csg_oracle_action_smeared_4d.restype = ctypes.c_double
    lib.csg_alg5_counts.argtypes = [_p_u64, _i64, _i64, _i64, _p_i64]
    lib.csg_alg5_counts.restype = None
    lib.csg_alg5_counts_rows.argtypes = [_p_u64, _i64, _i64, _i64, _i64, _i64, _p_i64,
                                         ctypes.POINTER(_i64)]
    lib.csg_alg5_counts_rows.restype = None
    lib.csg_oracle_link.argtypes = [ctypes.c_int, np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS"),
                                    _i64, _p_u8]
    lib.csg_oracle_link.restype = None
    lib.csg_oracle_link_dim.argtypes = [ctypes.c_int]
    lib.csg_oracle_link_dim.restype = ctypes.c_int
    _p_f64 = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
    lib.csg_dominance2d_counts.argtypes = [_p_f64, _i64, _i64, _p_i64]
    lib.csg_dominance2d_counts.restype = ctypes.c_int
    lib.csg_dominance2d_counts_rows.argtypes = [_p_f64, _i64, _i64, _i64, _i64, _p_i64]
    lib.csg_dominance2d_counts_rows.restype = ctypes.c_int
    lib.csg_dominance2d_relations.argtypes = [_p_f64, _i64]
    lib.csg_dominance2d_relations.restype = _i64
    lib.csg_alg5_threads.argtypes = []
    lib.csg_alg5_threads.restype = ctypes.c_int
    _lib = lib
    return lib


def _check_bits(bits, N):
    bits = np.ascontiguousarray(bits, dtype=np.uint64)
    assert bits.ndim == 2 and bits.shape[0] >= N and bits.shape[1] * 64 >= N, bits.shape
    return bits


def expand(bits, N):
    """Packed relation matrix -> N x N byte matrix (PAPER.md:163-169 layout)."""
    bits = _check_bits(bits, N)
    B = np.zeros((N, N), dtype=np.uint8)
    if N > 0:
        _load().csg_oracle_expand(bits, N, bits.shape[1], B)
    return B


def counts_plain(B, kmax):
    """Naive action algorithm on a byte matrix: counts[0..kmax]."""
    B = np.ascontiguousarray(B, dtype=np.uint8)
    N = B.shape[0]
    assert B.shape == (N, N)
    counts = np.zeros(kmax + 1, dtype=np.int64)
    _load().csg_oracle_counts(B, N, kmax, counts)
    return counts


def counts_from_bits(bits, N, kmax):
    """expand() then counts_plain(): the oracle on the same packed bitset the GPU gets."""
    return counts_plain(expand(bits, N), kmax)


def pair_interval(bits, N, i, j):
    """n_ij for one pair, bit by bit from the packed matrix; -1 if unrelated."""
    bits = _check_bits(bits, N)
    return int(_load().csg_oracle_pair(bits, N, bits.shape[1], int(i), int(j)))


def action_local(dim, N, counts):
    """Eq. 4 (dim=2) or the d=4 BD combination (reading A8)."""
    counts = np.ascontiguousarray(counts, dtype=np.int64)
    need = 3 if dim == 2 else 4
    if counts.shape[0] < need:
        counts = np.concatenate([counts, np.zeros(need - counts.shape[0], dtype=np.int64)])
    return float(_load().csg_oracle_action_local(int(dim), int(N), counts))


def f2(k, eps):
    """Smearing weight f_2(k, eps) of Eq. 5."""
    return float(_load().csg_oracle_f2(int(k), float(eps)))


def action_smeared_2d(N, counts, eps):
    """Eq. 5 over counts[0..len-1]; returns (S_eps, abs_scale)."""
    counts = np.ascontiguousarray(counts, dtype=np.int64)
    scale = ctypes.c_double(0.0)
    s = _load().csg_oracle_action_smeared_2d(int(N), counts.shape[0] - 1, counts, float(eps),
                                             ctypes.byref(scale))
    return float(s), float(scale.value)


def f4(k, eps):
    """Smearing weight f_4(k, eps) of the d=4 action (NOT IN PAPER; reading A9)."""
    return float(_load().csg_oracle_f4(int(k), float(eps)))


def action_smeared_4d(N, counts, eps):
    """d=4 smeared action (reading A9) over counts[0..len-1]; returns (S_eps, abs_scale)."""
    counts = np.ascontiguousarray(counts, dtype=np.int64)
    scale = ctypes.c_double(0.0)
    s = _load().csg_oracle_action_smeared_4d(int(N), counts.shape[0] - 1, counts, float(eps), ctypes.byref(scale))
    return float(s), float(scale.value)


def alg5_counts(bits, N, kmax):
    """Algorithm 5 on the packed matrix, all host threads."""
    bits = _check_bits(bits, N)
    counts = np.zeros(kmax + 1, dtype=np.int64)
    _load().csg_alg5_counts(bits, N, bits.shape[1], kmax, counts)
    return counts


def alg5_counts_rows(bits, N, kmax, row_begin, row_end):
    """Algorithm 5 restricted to first elements i in [row_begin,row_end); returns (counts, triple_tests)."""
    bits = _check_bits(bits, N)
    counts = np.zeros(kmax + 1, dtype=np.int64)
    tests = _i64(0)
    _load().csg_alg5_counts_rows(bits, N, bits.shape[1], kmax, int(row_begin), int(row_end), counts,
                                 ctypes.byref(tests))
    return counts, int(tests.value)


def dominance2d_counts(coords, kmax):
    """Interval abundances of a random 2D order straight from its (u, v) coordinates: n_ab = number of points
    strictly inside the rectangle spanned by a related pair (PAPER.md:395 for a 2D order; SURVEY pin P6).  No
    relation matrix is involved.  coords: (N, 2), any order, no repeated u or v."""
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    assert coords.ndim == 2 and coords.shape[1] == 2, coords.shape
    counts = np.zeros(kmax + 1, dtype=np.int64)
    rc = _load().csg_dominance2d_counts(coords, coords.shape[0], int(kmax), counts)
    if rc != 0:
        raise ValueError("dominance2d_counts: %s" % ("repeated coordinate" if rc == -1 else "out of memory"))
    return counts


def dominance2d_counts_rows(coords, kmax, row_begin, row_end):
    """dominance2d_counts restricted to related pairs whose lower element is one of coords[row_begin:row_end]
    (the split by first element of alg5_counts_rows when coords are in time order)."""
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    assert coords.ndim == 2 and coords.shape[1] == 2, coords.shape
    counts = np.zeros(kmax + 1, dtype=np.int64)
    rc = _load().csg_dominance2d_counts_rows(coords, coords.shape[0], int(kmax), int(row_begin), int(row_end), counts)
    if rc != 0:
        raise ValueError("dominance2d_counts_rows: %s" % ("repeated coordinate" if rc == -1 else "out of memory"))
    return counts


def dominance2d_relations(coords):
    """Number of related pairs of a random 2D order = C(N,2) - inversions (SURVEY pin P5), from coordinates."""
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    assert coords.ndim == 2 and coords.shape[1] == 2, coords.shape
    r = int(_load().csg_dominance2d_relations(coords, coords.shape[0]))
    if r < 0:
        raise ValueError("dominance2d_relations: %s" % ("repeated coordinate" if r == -1 else "out of memory"))
    return r


def alg5_threads():
    return int(_load().csg_alg5_threads())


GEOM_MINKOWSKI_2D, GEOM_MINKOWSKI_4D, GEOM_DESITTER_2D = 0, 1, 2


def link(geometry, coords):
    """Dense linking (de Sitter test PAPER.md:465): time-sorted coordinates (N, dim) ->
    symmetric N x N byte matrix, zero diagonal."""
    lib = _load()
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    N, dim = coords.shape
    assert dim == lib.csg_oracle_link_dim(int(geometry))
    B = np.zeros((N, N), dtype=np.uint8)
    if N:
        lib.csg_oracle_link(int(geometry), coords, N, B)
    return B
