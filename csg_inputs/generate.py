"""ctypes front end of csg_inputs/gen.c plus a few tiny structured posets for tests."""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libcsggen.so")
_SRC = os.path.join(_HERE, "gen.c")
_lib = None

# BASELINE.json "configs", in order.  kmax = highest interval size kept; eps = 1.0 means the local action.
_SEED0 = 170903013
CONFIGS = [
    dict(name="cfg0_2d_1024", dim=2, N=1024, eps=1.0, kmax=3, seed=_SEED0 + 0),
    dict(name="cfg1_2d_16384", dim=2, N=16384, eps=1.0, kmax=3, seed=_SEED0 + 1),
    dict(name="cfg2_4d_65536", dim=4, N=65536, eps=1.0, kmax=3, seed=_SEED0 + 2),
    dict(name="cfg3_4d_131072", dim=4, N=131072, eps=1.0, kmax=3, seed=_SEED0 + 3),
    dict(name="cfg4_2d_262144_smeared", dim=2, N=262144, eps=0.1, kmax=262142, seed=_SEED0 + 4),
    # not a BASELINE.json config: the paper's own benchmark workload (Fig. 4): (1+1) de Sitter slab,
    # eta0 = 0.5, largest N of its range, smeared action with eps = 2^-6
    dict(name="paper_ds2_131072_smeared", dim=2, N=131072, eps=2.0 ** -6, kmax=131070, seed=_SEED0 + 5,
         geometry="ds2", eta0=0.5),
]


def make_config(cfg, seed=None):
    """(coords, bits) of a CONFIGS entry (flat diamond or de Sitter slab)."""
    seed = cfg["seed"] if seed is None else seed
    if cfg.get("geometry") == "ds2":
        return make_de_sitter(cfg["N"], seed, cfg.get("eta0", 0.5))
    return make_causet(cfg["dim"], cfg["N"], seed)

_p_f64 = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_p_u64 = np.ctypeslib.ndpointer(dtype=np.uint64, flags="C_CONTIGUOUS")


def build(force=False):
    if not force and os.path.exists(_LIB_PATH) and os.path.getmtime(_LIB_PATH) >= os.path.getmtime(_SRC):
        return _LIB_PATH
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB_PATH, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB_PATH)
        lib.csg_gen_stride_words.argtypes = [ctypes.c_int64]
        lib.csg_gen_stride_words.restype = ctypes.c_int64
        for name in ("csg_gen_coords_2d", "csg_gen_coords_4d"):
            f = getattr(lib, name)
            f.argtypes = [ctypes.c_uint64, ctypes.c_int64, _p_f64]
            f.restype = ctypes.c_int
        for name in ("csg_gen_relations_2d", "csg_gen_relations_4d"):
            f = getattr(lib, name)
            f.argtypes = [_p_f64, ctypes.c_int64, _p_u64]
            f.restype = ctypes.c_int
        lib.csg_gen_coords_ds2.argtypes = [ctypes.c_uint64, ctypes.c_int64, ctypes.c_double, _p_f64]
        lib.csg_gen_coords_ds2.restype = ctypes.c_int
        lib.csg_gen_relations_ds2.argtypes = [_p_f64, ctypes.c_int64, _p_u64]
        lib.csg_gen_relations_ds2.restype = ctypes.c_int
        lib.csg_gen_hash.argtypes = [_p_u64, ctypes.c_int64]
        lib.csg_gen_hash.restype = ctypes.c_uint64
        _lib = lib
    return _lib


def stride_words(N):
    """Row stride in 64-bit words: rows are 256-bit aligned."""
    return 4 * ((int(N) + 255) // 256)


def sprinkle(dim, N, seed):
    """Time-sorted coordinates, shape (N, dim): (u, v) for dim=2, (t, x, y, z) for dim=4."""
    assert dim in (2, 4)
    coords = np.zeros((N, dim), dtype=np.float64)
    fn = _load().csg_gen_coords_2d if dim == 2 else _load().csg_gen_coords_4d
    if N > 0 and fn(int(seed), int(N), coords) != 0:
        raise MemoryError("sprinkle")
    return coords


def relations_from_coords(coords):
    """Packed symmetric relation matrix, shape (N, stride_words(N)) uint64."""
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    N, dim = coords.shape
    bits = np.zeros((N, stride_words(N)), dtype=np.uint64)
    fn = _load().csg_gen_relations_2d if dim == 2 else _load().csg_gen_relations_4d
    if N > 0:
        fn(coords, N, bits)
    return bits


def make_causet(dim, N, seed):
    """(coords, bits) of a seeded sprinkling into the flat causal diamond."""
    coords = sprinkle(dim, N, seed)
    return coords, relations_from_coords(coords)


def sprinkle_de_sitter(N, seed, eta0=0.5):
    """(1+1) de Sitter slab |eta| <= eta0: conformal-time-sorted (eta, theta), shape (N, 2)."""
    coords = np.zeros((N, 2), dtype=np.float64)
    if N > 0 and _load().csg_gen_coords_ds2(int(seed), int(N), float(eta0), coords) != 0:
        raise MemoryError("sprinkle_de_sitter")
    return coords


def relations_de_sitter(coords):
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    N = coords.shape[0]
    bits = np.zeros((N, stride_words(N)), dtype=np.uint64)
    if N > 0:
        _load().csg_gen_relations_ds2(coords, N, bits)
    return bits


def make_de_sitter(N, seed, eta0=0.5):
    """(coords, bits) of a seeded sprinkling into the (1+1) de Sitter slab, the paper's benchmark workload."""
    coords = sprinkle_de_sitter(N, seed, eta0)
    return coords, relations_de_sitter(coords)


def bits_hash(bits):
    b = np.ascontiguousarray(bits, dtype=np.uint64)
    return int(_load().csg_gen_hash(b.reshape(-1), b.size))


def pack_dense(upper):
    """Pack a dense 0/1 matrix: entry (i, j), i<j, of `upper` says i precedes j.  The result is the
    symmetric, zero-diagonal packed layout the library takes.  For small hand-built posets in tests."""
    upper = np.triu(np.asarray(upper) != 0, 1)
    N = upper.shape[0]
    sym = upper | upper.T
    W = stride_words(N)
    padded = np.zeros((N, W * 64), dtype=np.uint8)
    padded[:, :N] = sym
    by = np.packbits(padded, axis=1, bitorder="little")
    return np.ascontiguousarray(by).view(np.uint64).reshape(N, W)


def random_poset_bits(N, p, seed, transitive=True):
    """Random order on 0..N-1 compatible with the index order: each i<j related with probability p,
    optionally transitively closed.  Returns (upper bool matrix, packed bits)."""
    rng = np.random.default_rng(seed)
    up = np.triu(rng.random((N, N)) < p, 1)
    if transitive:
        for k in range(N):
            up |= np.outer(up[:, k], up[k, :])
        up = np.triu(up, 1)
    return up, pack_dense(up)
