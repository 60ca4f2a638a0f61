"""Block-sparse K sweep of the fp4 tensor kernel (include/csg.h: csg_set_sparse, csg_block_occupancy): the occupancy
pass against numpy on the same bitset, and the action with the sweep forced on against the oracle on relation
matrices that have empty 256 x 256 blocks in every position a tile can meet them (first stages, last stages, the
middle of the sweep, whole tiles dead, nothing alive at all).  Results must never depend on the sweep."""
import numpy as np
import pytest

import csg_inputs
import oracle

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def csg():
    import paper_1709_03013_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    if m._build.needs_build():
        m.build()
    m.load()
    yield m
    m.csg_set_variant(m.VARIANT_AUTO)
    m.csg_set_sparse(m.SPARSE_AUTO)


def block_sparse_poset(N, density, keep_prob, seed):
    """Index-compatible random relation matrix (not transitively closed: the definition does not need it, DESIGN.md
    A12, and a closure would refill the blocks) whose 256 x 256 blocks (I, K), I <= K, survive with probability
    keep_prob, and of the survivors' 256 x 128 and 128 x 256 half-blocks another quarter is emptied.  Returns the packed bitset and the dense upper-triangular 0/1 matrix."""
    rng = np.random.default_rng(seed)
    U = np.triu(rng.random((N, N)) < density, 1)
    nB = (N + 255) // 256
    keep = rng.random((nB, nB)) < keep_prob
    U &= np.kron(keep, np.ones((256, 256), dtype=bool))[:N, :N]
    U &= np.kron(rng.random((nB, 2 * nB)) < 0.75, np.ones((256, 128), dtype=bool))[:N, :N]
    U &= np.kron(rng.random((2 * nB, nB)) < 0.75, np.ones((128, 256), dtype=bool))[:N, :N]
    return csg_inputs.pack_dense(U.astype(np.uint8)), U


def occupancy_numpy(U_sym, N):
    nB = (N + 255) // 256
    pad = np.zeros((256 * nB, 256 * nB), dtype=bool)
    pad[:N, :N] = U_sym
    return pad.reshape(nB, 256, nB, 256).any(axis=(1, 3))


def unpack_occ(occ, nB):
    w = occ.cpu().numpy().view(np.uint32)
    bits = ((w[:, :, None] >> np.arange(32, dtype=np.uint32)[None, None, :]) & 1).astype(bool).reshape(w.shape[0], -1)
    assert not bits[:, nB:].any(), "padding words of the occupancy map must be zero"
    return bits[:, :nB]


@pytest.mark.parametrize("N", [1, 255, 256, 257, 1000, 4097, 8192 + 300, 33000])
def test_block_occupancy_equals_numpy(csg, N):
    rng = np.random.default_rng(N)
    nB = (N + 255) // 256
    if N <= 4097:
        bits, U = block_sparse_poset(N, 0.02, 0.5, N)
        sym = U | U.T
        want = occupancy_numpy(sym, N)
    else:                                # large: a handful of single relations at known places
        stride = csg_inputs.stride_words(N)
        bits = np.zeros((N, stride), dtype=np.uint64)
        want = np.zeros((nB, nB), dtype=bool)
        for _ in range(200):
            i, j = sorted(int(x) for x in rng.integers(0, N, 2))
            if i == j:
                continue
            bits[i, j // 64] |= np.uint64(1) << np.uint64(j % 64)
            bits[j, i // 64] |= np.uint64(1) << np.uint64(i % 64)
            want[i // 256, j // 256] = want[j // 256, i // 256] = True
    occ = csg.csg_block_occupancy(csg.to_device(bits), N)
    torch.cuda.synchronize()
    assert occ.shape == (nB, csg.csg_occupancy_stride_words(N))
    assert (unpack_occ(occ, nB) == want).all()


@pytest.mark.parametrize("N,density,keep,seed", [
    (700, 0.05, 0.5, 1), (1025, 0.03, 0.4, 2), (2049, 0.02, 0.3, 3), (2600, 0.02, 0.6, 4), (3000, 0.01, 0.15, 5),
    (2560, 0.02, 0.0, 6),                # nothing alive at all
    (2304, 0.02, 1.0, 7),                # nothing dead
])
def test_sparse_sweep_equals_oracle(csg, N, density, keep, seed):
    bits, _ = block_sparse_poset(N, density, keep, seed)
    kmax = N - 2
    want = oracle.counts_from_bits(bits, N, kmax) if N <= 1200 else oracle.alg5_counts(bits, N, kmax)
    d = csg.to_device(bits)
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    try:
        for mode in (csg.SPARSE_ON, csg.SPARSE_OFF, csg.SPARSE_ON):
            csg.csg_set_sparse(mode)
            for throttle in (csg.THROTTLE_OFF, csg.THROTTLE_ON):
                csg.csg_set_throttle(throttle)
                c, S = csg.csg_action(d, N, 2, 0.25, kmax)
                torch.cuda.synchronize()
                got = c.cpu().numpy()
                assert (got == want).all(), (mode, throttle, np.nonzero(got != want)[0][:10])
                s_want, scale = oracle.action_smeared_2d(N, want, 0.25)
                assert abs(float(S.item()) - s_want) <= 1e-12 * scale
    finally:
        csg.csg_set_throttle(csg.THROTTLE_AUTO)
        csg.csg_set_sparse(csg.SPARSE_AUTO)
        csg.csg_set_variant(csg.VARIANT_AUTO)


def test_sparse_sweep_single_populated_block(csg):
    """Only block (0, 5) of the matrix holds relations: tile (0, 5) has related pairs and not one live stage, so every one
    of them has n_ij = 0 -- the kernel must still run one (all-zero) group to clear its accumulators."""
    N = 6 * 256
    rng = np.random.default_rng(11)
    U = np.zeros((N, N), dtype=bool)
    U[0:256, 5 * 256:6 * 256] = rng.random((256, 256)) < 0.3
    bits = csg_inputs.pack_dense(U.astype(np.uint8))
    want = oracle.counts_from_bits(bits, N, N - 2)
    assert want[0] == U.sum() and want[1:].sum() == 0
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    csg.csg_set_sparse(csg.SPARSE_ON)
    try:
        for _ in range(3):                     # stale accumulators of an earlier tile would show on a repeat
            c, _ = csg.csg_action(csg.to_device(bits), N, 2, 0.5, N - 2)
            torch.cuda.synchronize()
            assert (c.cpu().numpy() == want).all()
    finally:
        csg.csg_set_sparse(csg.SPARSE_AUTO)
        csg.csg_set_variant(csg.VARIANT_AUTO)


@pytest.mark.parametrize("N,keep,seed", [(1300, 0.5, 1), (2049, 0.3, 2)])
def test_sparse_tile_dump_pair_by_pair(csg, N, keep, seed):
    """Every n_ij of every tile from the tensor kernel with the sweep forced on, against U @ U."""
    bits, U = block_sparse_poset(N, 0.03, keep, seed)
    Ui = U.astype(np.int64)
    want = np.where(Ui == 1, Ui @ Ui, -1)
    nB = (N + 255) // 256
    tiles = [(I, J) for I in range(nB) for J in range(I, nB)]
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    csg.csg_set_sparse(csg.SPARSE_ON)
    try:
        dump = csg.csg_tile_interval_sizes(csg.to_device(bits), N, tiles).cpu().numpy()
    finally:
        csg.csg_set_sparse(csg.SPARSE_AUTO)
        csg.csg_set_variant(csg.VARIANT_AUTO)
    padded = np.full((256 * nB, 256 * nB), -1, dtype=np.int64)
    padded[:N, :N] = want
    for t, (I, J) in enumerate(tiles):
        assert (dump[t] == padded[256 * I:256 * I + 256, 256 * J:256 * J + 256]).all(), (I, J)


@pytest.mark.parametrize("dim,N,kmax", [(4, 20001, 3), (4, 16384, 16382), (2, 9001, 8999)])
def test_sparse_sweep_sprinkled_sets(csg, dim, N, kmax):
    """Sprinkled sets at sizes that take the patch schedule (several rounds per cluster), sweep forced on, with shards."""
    _, bits = csg_inputs.make_causet(dim, N, 77 + N)
    want = oracle.alg5_counts(bits, N, kmax)
    d = csg.to_device(bits)
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    csg.csg_set_sparse(csg.SPARSE_ON)
    try:
        for _ in range(2):
            c, S = csg.csg_action(d, N, dim, 1.0, kmax)
            torch.cuda.synchronize()
            assert (c.cpu().numpy() == want).all()
            assert float(S.item()) == oracle.action_local(dim, N, want)
        total = np.zeros(kmax + 1, dtype=np.int64)
        for s in range(3):
            total += csg.csg_action_partial(d, N, kmax, s, 3).cpu().numpy()
        assert (total == want).all()
    finally:
        csg.csg_set_sparse(csg.SPARSE_AUTO)
        csg.csg_set_variant(csg.VARIANT_AUTO)


@pytest.mark.parametrize("pipeline", ["auto", "chunked"])
@pytest.mark.parametrize("dim,N,kmax", [(4, 20001, 3), (2, 16384, 16382), (4, 33000, 3)])
def test_sparse_sweep_in_the_host_pipeline(csg, dim, N, kmax, pipeline):
    """csg_action_host with the sweep forced on: the copy stream marks the occupancy rows of every chunk behind its copy,
    while the (gated or chunked) interval kernel already runs; pinned and pageable host memory, repeated calls."""
    _, bits = csg_inputs.make_causet(dim, N, 5 + N)
    want = oracle.alg5_counts(bits, N, kmax)
    pinned = torch.from_numpy(bits.view(np.int64)).pin_memory()
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    csg.csg_set_sparse(csg.SPARSE_ON)
    csg.csg_set_host_pipeline(csg.HOST_PIPELINE_CHUNKED if pipeline == "chunked" else csg.HOST_PIPELINE_AUTO)
    try:
        for host in (pinned, bits, pinned):
            c, S = csg.csg_action_host(host, N, dim, 1.0, kmax)
            assert (np.asarray(c) == want).all()
            assert S == oracle.action_local(dim, N, want)
    finally:
        csg.csg_set_host_pipeline(csg.HOST_PIPELINE_AUTO)
        csg.csg_set_sparse(csg.SPARSE_AUTO)
        csg.csg_set_variant(csg.VARIANT_AUTO)


def test_sparse_and_batched_launches_in_a_cuda_graph(csg):
    """After one warm-up call per size the block-sparse call (occupancy kernel + interval kernel; its occupancy map comes
    from a ring that is allocated as a whole by the warm-up) and the batched call (one persistent launch over all sets)
    only enqueue stream-ordered work: captured in a CUDA graph and replayed twice, with other calls in between."""
    N, dim, kmax = 5000, 4, 3
    sets = [csg_inputs.make_causet(dim, N, 40 + b)[1] for b in range(3)]
    want = [oracle.alg5_counts(b, N, kmax) for b in sets]
    d = [csg.to_device(b) for b in sets]
    nb, Nb = 12, 700
    small = np.stack([csg_inputs.make_causet(2, Nb, 300 + b)[1] for b in range(nb)])
    d_small = csg.to_device(small)
    want_small = [oracle.counts_from_bits(small[b], Nb, 3) for b in range(nb)]
    other = csg_inputs.make_causet(dim, 1300, 77)[1]
    d_other, want_other = csg.to_device(other), oracle.alg5_counts(other, 1300, kmax)
    counts = [torch.zeros(kmax + 1, dtype=torch.int64, device="cuda") for _ in sets]
    S = [torch.zeros(1, dtype=torch.float64, device="cuda") for _ in sets]
    bc = torch.zeros((nb, 4), dtype=torch.int64, device="cuda")
    bS = torch.zeros(nb, dtype=torch.float64, device="cuda")
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    csg.csg_set_sparse(csg.SPARSE_ON)
    try:
        csg.csg_action(d[0], N, dim, 1.0, kmax, counts[0], S[0])                     # warm-ups outside the capture
        csg.csg_action_batch(d_small, Nb, nb, 2, 1.0, 3, bc, bS)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            for b in range(3):
                csg.csg_action(d[b], N, dim, 1.0, kmax, counts[b], S[b])
            csg.csg_action_batch(d_small, Nb, nb, 2, 1.0, 3, bc, bS)
        for rep in range(2):
            for c in counts:
                c.fill_(-1)
            bc.fill_(-1)
            graph.replay()
            torch.cuda.synchronize()
            for b in range(3):
                assert (counts[b].cpu().numpy() == want[b]).all(), (rep, b)
                assert float(S[b].item()) == oracle.action_local(dim, N, want[b])
            got = bc.cpu().numpy()
            for b in range(nb):
                assert (got[b] == want_small[b]).all(), (rep, b)
            c2, _ = csg.csg_action(d_other, 1300, dim, 1.0, kmax)                       # another size in between
            torch.cuda.synchronize()
            assert (c2.cpu().numpy() == want_other).all()
    finally:
        csg.csg_set_sparse(csg.SPARSE_AUTO)
        csg.csg_set_variant(csg.VARIANT_AUTO)


FIRST_CALL_SCRIPT = r"""
import sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch
import csg_inputs, paper_1709_03013_b200 as csg
csg.load()
N, dim, kmax = 16384, 4, 3
_, bits = csg_inputs.make_causet(dim, N, 4711)
csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
csg.csg_set_sparse(csg.SPARSE_ON)
c_host, S_host = csg.csg_action_host(bits, N, dim, 1.0, kmax)          # the FIRST call of this process into the library
c_dev, S_dev = csg.csg_action(csg.to_device(bits), N, dim, 1.0, kmax)
torch.cuda.synchronize()
assert (np.asarray(c_host) == c_dev.cpu().numpy()).all() and S_host == float(S_dev.item())
print("FIRST_CALL_OK", [int(x) for x in c_host])
"""


def test_host_pipeline_as_the_first_call_of_a_process(csg):
    """csg_action_host with the block-sparse sweep as the very first library call of a fresh process: the occupancy
    kernels it launches while the gated interval kernel already waits for the copies must have been loaded before that
    kernel starts (CUDA loads kernels lazily, loading may synchronise the context: this call once hung for good).  Run
    in a subprocess under a timeout, so that a hang fails instead of stalling the suite."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", FIRST_CALL_SCRIPT, root], capture_output=True, text=True, timeout=240)
    assert r.returncode == 0 and "FIRST_CALL_OK" in r.stdout, (r.returncode, r.stdout[-500:], r.stderr[-1500:])
    _, bits = csg_inputs.make_causet(4, 16384, 4711)
    want = oracle.alg5_counts(bits, 16384, 3)
    assert str([int(x) for x in want]) in r.stdout
