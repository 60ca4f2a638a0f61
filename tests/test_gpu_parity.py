"""Parity of the CUDA path (through the C ABI) with the oracle, element by element, on the same seeded
inputs.  Counts are int64 and must match bit for bit; the local action is an exact integer times a constant
and must match exactly; the smeared action within 1e-12 of its term scale."""
import math

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


VARIANTS = [1, 2, 3]


def run_action(csg, bits, N, dim, eps, kmax, variant):
    csg.csg_set_variant(variant)
    counts, S = csg.csg_action(csg.to_device(bits), N, dim, eps, kmax)
    torch.cuda.synchronize()
    return counts.cpu().numpy(), float(S.item())


def reference_counts(bits, N, kmax):
    return oracle.counts_from_bits(bits, N, kmax) if N <= 1200 else oracle.alg5_counts(bits, N, kmax)


# --------------------------------------------------------------------------- small and ragged sizes
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("N", [1, 2, 3, 31, 63, 64, 65, 127, 128, 129, 255, 256, 257, 383, 385, 511, 513, 777, 1025])
def test_random_posets_full_histogram(csg, variant, N):
    for transitive in (True, False):
        _, bits = csg_inputs.random_poset_bits(N, min(0.5, 8.0 / max(N, 1) + 0.02), seed=N, transitive=transitive)
        kmax = max(N - 2, 3)
        want = oracle.counts_from_bits(bits, N, kmax)
        got, S = run_action(csg, bits, N, 2, 1.0, kmax, variant)
        assert (got == want).all(), (N, transitive, np.nonzero(got != want)[0][:10])
        assert S == oracle.action_local(2, N, want)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("dim,N,seed", [(2, 300, 1), (4, 300, 2), (2, 1500, 3), (4, 1500, 4), (4, 2600, 5), (2, 3000, 6)])
def test_sprinkled_local_action(csg, variant, dim, N, seed):
    _, bits = csg_inputs.make_causet(dim, N, seed)
    want = reference_counts(bits, N, 3)
    got, S = run_action(csg, bits, N, dim, 1.0, 3, variant)
    assert (got == want).all(), (got, want)
    assert S == oracle.action_local(dim, N, want)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("N,eps", [(700, 0.1), (1500, 2.0 ** -6), (2100, 0.5)])
def test_smeared_action_full_histogram(csg, variant, N, eps):
    _, bits = csg_inputs.make_causet(2, N, 40 + N)
    want = reference_counts(bits, N, N - 2)
    got, S = run_action(csg, bits, N, 2, eps, N - 2, variant)
    assert (got == want).all()
    s_want, scale = oracle.action_smeared_2d(N, want, eps)
    assert abs(S - s_want) <= 1e-12 * scale, (S, s_want, scale)


@pytest.mark.parametrize("variant", VARIANTS)
def test_kmax_truncation_and_dense_chain(csg, variant):
    """Total order of 600 elements: N_k = N-1-k (largest possible interval sizes); kmax cuts, never clamps."""
    N = 600
    bits = csg_inputs.pack_dense(np.triu(np.ones((N, N)), 1))
    got, S = run_action(csg, bits, N, 2, 1.0, N - 2, variant)
    assert (got == N - 1 - np.arange(N - 1)).all() and S == 2.0 * N
    got, _ = run_action(csg, bits, N, 4, 1.0, 10, variant)
    assert (got == N - 1 - np.arange(11)).all()


@pytest.mark.parametrize("variant", VARIANTS)
def test_empty_relation_and_dirty_diagonal(csg, variant):
    N = 500
    got, S = run_action(csg, csg_inputs.pack_dense(np.zeros((N, N))), N, 4, 1.0, 3, variant)
    assert got.sum() == 0 and S == (4.0 / math.sqrt(6.0)) * N
    up, bits = csg_inputs.random_poset_bits(N, 0.05, seed=3)
    want = oracle.counts_from_bits(bits, N, N - 2)
    dirty = bits.copy()
    for r in range(N):
        dirty[r, r // 64] |= np.uint64(1) << np.uint64(r % 64)
    got, _ = run_action(csg, dirty, N, 2, 1.0, N - 2, variant)
    assert (got == want).all()


def test_repeat_calls_are_deterministic_and_overwrite(csg):
    _, bits = csg_inputs.make_causet(2, 2500, 9)
    d = csg.to_device(bits)
    csg.csg_set_variant(csg.VARIANT_TENSOR)
    counts = torch.full((2499,), 77, dtype=torch.int64, device="cuda")
    S = torch.zeros(1, dtype=torch.float64, device="cuda")
    outs = []
    for _ in range(3):
        csg.csg_action(d, 2500, 2, 0.1, 2498, counts, S)
        torch.cuda.synchronize()
        outs.append((counts.cpu().numpy().copy(), S.item()))
    assert all((o[0] == outs[0][0]).all() and o[1] == outs[0][1] for o in outs)
    assert (outs[0][0] == oracle.alg5_counts(bits, 2500, 2498)).all()


def test_host_entry_point(csg):
    _, bits = csg_inputs.make_causet(4, 2300, 10)
    csg.csg_set_variant(csg.VARIANT_AUTO)
    counts, S = csg.csg_action_host(bits, 2300, 4, 1.0, 3)
    want = oracle.alg5_counts(bits, 2300, 3)
    assert (counts == want).all() and S == oracle.action_local(4, 2300, want)
    pinned = torch.from_numpy(bits.view(np.int64)).pin_memory()
    counts2, S2 = csg.csg_action_host(pinned, 2300, 4, 1.0, 3)
    assert (counts2 == want).all() and S2 == S


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("dim,N,eps,nshards", [(4, 2600, 1.0, 2), (2, 1900, 0.25, 3), (2, 300, 1.0, 8)])
def test_tile_shards_sum_to_the_whole(csg, variant, dim, N, eps, nshards):
    """csg_action_partial over every shard, summed (what the all-reduce does), then csg_action_finish ==
    csg_action == oracle."""
    _, bits = csg_inputs.make_causet(dim, N, 70 + N)
    kmax = N - 2
    want = reference_counts(bits, N, kmax)
    d = csg.to_device(bits)
    csg.csg_set_variant(variant)
    total = torch.zeros(kmax + 1, dtype=torch.int64, device="cuda")
    for s in range(nshards):
        total += csg.csg_action_partial(d, N, kmax, s, nshards)
    S = csg.csg_action_finish(total, N, dim, eps, kmax)
    whole, S_whole = csg.csg_action(d, N, dim, eps, kmax)
    torch.cuda.synchronize()
    assert (total.cpu().numpy() == want).all()
    assert (whole.cpu().numpy() == want).all()
    assert float(S.item()) == float(S_whole.item())
    if eps == 1.0:
        assert float(S.item()) == oracle.action_local(dim, N, want)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("N,eps", [(900, 0.25), (2300, 2.0 ** -4)])
def test_smeared_action_4d(csg, variant, N, eps):
    """Reading A9 (not in the paper): d=4 smeared action from the full histogram."""
    _, bits = csg_inputs.make_causet(4, N, 90 + N)
    want = reference_counts(bits, N, N - 2)
    got, S = run_action(csg, bits, N, 4, eps, N - 2, variant)
    assert (got == want).all()
    s_want, scale = oracle.action_smeared_4d(N, want, eps)
    assert abs(S - s_want) <= 1e-12 * scale + 1e-15 * abs(s_want), (S, s_want, scale)


@pytest.mark.parametrize("variant", [0, 2])
@pytest.mark.parametrize("dim,N,batch,eps", [(2, 1, 3, 1.0), (2, 100, 9, 0.3), (2, 200, 7, 1.0), (4, 1000, 5, 1.0), (2, 513, 40, 0.1),
                                               (4, 2200, 3, 1.0), (2, 2100, 2, 0.5), (2, 512, 150, 1.0), (4, 777, 33, 1.0),
                                               (2, 4100, 9, 1.0), (2, 129, 300, 1.0)])
def test_batch_of_causal_sets(csg, dim, N, batch, eps, variant):
    """csg_action_batch: every set of the batch equals the oracle and the single-set call.  One interval launch for the
    whole batch: the bitset kernel up to 128 elements, ONE persistent tensor launch over the tiles of all sets above
    (rows beyond a set's N inside its last 256-row block belong to the next set there, not to zero padding)."""
    csg.csg_set_variant(variant)
    kmax = 3 if eps == 1.0 else N - 2
    sets = [csg_inputs.make_causet(dim, N, 500 + 13 * b + N)[1] for b in range(batch)]
    d = csg.to_device(np.stack(sets))
    launches0 = csg.csg_launch_count()
    counts, S = csg.csg_action_batch(d, N, batch, dim, eps, kmax)
    torch.cuda.synchronize()
    launches = csg.csg_launch_count() - launches0
    tensor = csg.csg_effective_variant(2000) != csg.VARIANT_BITSET if variant else N > 128
    # bitset: one launch for the batch; tensor: one per power of two in the batch size; + the finishing kernel
    assert launches == (bin(batch).count("1") if tensor else 1) + 1
    counts, S = counts.cpu().numpy(), S.cpu().numpy()
    for b in range(batch):
        want = reference_counts(sets[b], N, kmax)
        assert (counts[b] == want).all(), b
        if eps == 1.0:
            assert S[b] == oracle.action_local(dim, N, np.concatenate([want, np.zeros(4, np.int64)]))
        else:
            s_want, scale = oracle.action_smeared_2d(N, want, eps)
            assert abs(S[b] - s_want) <= 1e-12 * scale
        c1, S1 = csg.csg_action(d[b], N, dim, eps, kmax)
        torch.cuda.synchronize()
        assert (c1.cpu().numpy() == counts[b]).all() and float(S1.item()) == S[b]


@pytest.mark.parametrize("dim,N,eps", [(2, 16384, 1.0), (4, 20001, 1.0), (2, 17000, 0.1)])
def test_host_entry_point_pipelined(csg, dim, N, eps):
    """Matrices of 32 MiB and more go to the device in row chunks, each chunk's tiles launched as it lands: same
    counts and S as the device-resident call and as Algorithm 5; pinned and pageable host memory; repeatable."""
    _, bits = csg_inputs.make_causet(dim, N, 4000 + N)
    kmax = 3 if eps == 1.0 else N - 2
    csg.csg_set_variant(csg.VARIANT_AUTO)
    want = oracle.alg5_counts(bits, N, kmax)
    counts, S = csg.csg_action_host(bits, N, dim, eps, kmax)                      # pageable
    assert (counts == want).all()
    pinned = torch.from_numpy(bits.view(np.int64)).pin_memory()
    for _ in range(2):
        counts2, S2 = csg.csg_action_host(pinned, N, dim, eps, kmax)
        assert (counts2 == want).all() and S2 == S
    c_dev, S_dev = csg.csg_action(csg.to_device(bits), N, dim, eps, kmax)
    torch.cuda.synchronize()
    assert (c_dev.cpu().numpy() == want).all() and float(S_dev.item()) == S
    csg.csg_set_variant(csg.VARIANT_TENSOR)                                       # int8 kind through the same path
    counts3, S3 = csg.csg_action_host(pinned, N, dim, eps, kmax)
    csg.csg_set_variant(csg.VARIANT_AUTO)
    assert (counts3 == want).all() and S3 == S


def test_sharded_call_on_one_rank(csg):
    """multigpu.csg_action_sharded without a process group is one shard of one: same result as csg_action."""
    from paper_1709_03013_b200 import multigpu
    _, bits = csg_inputs.make_causet(4, 2700, 12)
    d = csg.to_device(bits)
    csg.csg_set_variant(csg.VARIANT_AUTO)
    c1, S1 = multigpu.csg_action_sharded(d, 2700, 4, 1.0, 3)
    c2, S2 = csg.csg_action(d, 2700, 4, 1.0, 3)
    torch.cuda.synchronize()
    assert (c1.cpu().numpy() == oracle.alg5_counts(bits, 2700, 3)).all()
    assert torch.equal(c1, c2) and float(S1.item()) == float(S2.item())


def test_interval_sizes_hook(csg):
    N = 3000
    _, bits = csg_inputs.make_causet(4, N, 11)
    rng = np.random.default_rng(0)
    pairs = rng.integers(0, N, size=(4000, 2))
    pairs = np.concatenate([pairs, [[0, N - 1], [5, 5], [9, 3], [N - 2, N - 1], [0, 1], [63, 64], [64, 127]]])
    got = csg.csg_interval_sizes(csg.to_device(bits), N, torch.from_numpy(pairs.astype(np.int64)).cuda())
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    for (i, j), n in zip(pairs, got):
        assert n == oracle.pair_interval(bits, N, i, j), (i, j)


def test_error_codes_on_device(csg):
    d = torch.zeros(64, dtype=torch.int64, device="cuda")
    with pytest.raises(csg.CsgError) as e:
        csg._check(csg.load().csg_action(d.data_ptr() + 8, 8, 2, 1.0, 3, d.data_ptr(), d.data_ptr(), None))
    assert e.value.code == -3
    with pytest.raises(csg.CsgError) as e:
        csg._check(csg.load().csg_action(None, 8, 2, 1.0, 3, d.data_ptr(), d.data_ptr(), None))
    assert e.value.code == -1


# --------------------------------------------------------------------------- BASELINE.json configs
def degree_invariants(bits, N):
    """#relations and sum_k in_k*out_k from row popcounts (O(N^2/64), no N^3 code): for a transitive set the
    second equals the number of 3-chains = sum_k k N_k (pin P4)."""
    W = bits.shape[1]
    indeg = np.zeros(N, np.int64)
    outdeg = np.zeros(N, np.int64)
    cols = np.arange(W)
    for r0 in range(0, N, 2048):
        blk = bits[r0:r0 + 2048]
        pc = np.bitwise_count(blk).astype(np.int64)
        rows = np.arange(r0, r0 + blk.shape[0])
        wi = rows // 64
        below = (pc * (cols[None, :] < wi[:, None])).sum(1)
        own = blk[np.arange(blk.shape[0]), wi]
        lowmask = (np.uint64(1) << (rows % 64).astype(np.uint64)) - np.uint64(1)
        below += np.bitwise_count(own & lowmask).astype(np.int64)
        indeg[rows] = below
        outdeg[rows] = pc.sum(1) - below
    return int(outdeg.sum()), int((indeg * outdeg).sum())


def golden_histogram(name):
    """Line of tests/golden/config_histograms.txt for this config (written by tests/golden/make_config_goldens.py,
    which calls only the oracle), or None."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config_histograms.txt")
    for ln in open(path):
        f = ln.split()
        if f and f[0] == name:
            return dict(N=int(f[1]), kmax=int(f[2]), bits_hash=int(f[3], 16), sha256=f[4], total=int(f[5]),
                        head=[int(x) for x in f[6:14]])
    return None


def check_config(csg, cfg, full_reference):
    N, dim = cfg["N"], cfg["dim"]
    coords, bits = csg_inputs.make_causet(dim, N, cfg["seed"])
    d = csg.to_device(bits)
    csg.csg_set_variant(csg.VARIANT_AUTO)
    # (1) the configuration as benchmarked
    counts, S = csg.csg_action(d, N, dim, cfg["eps"], cfg["kmax"])
    torch.cuda.synchronize()
    counts = counts.cpu().numpy()
    # (2) full histogram through the same launch configuration: properties that hold at any size
    full, _ = csg.csg_action(d, N, 2, 1.0, N - 2)
    torch.cuda.synchronize()
    full = full.cpu().numpy()
    assert (full[:cfg["kmax"] + 1] == counts).all()
    nrel, chains = degree_invariants(bits, N)
    assert full.sum() == nrel                                         # I1
    if dim == 2:
        assert full.sum() == oracle.dominance2d_relations(coords)     # P5: C(N,2) - inversions, from the coordinates
    assert int((np.arange(N - 1, dtype=object) * full.astype(object)).sum()) == chains   # I2 = I3
    # (2b) the tile shards of the multi-GPU path (patch schedule at these sizes) add up to the same histogram
    parts = sum(csg.csg_action_partial(d, N, cfg["kmax"], s, 3) for s in range(3))
    torch.cuda.synchronize()
    assert (parts.cpu().numpy() == counts).all()
    # (3) sampled outputs the oracle computes one by one, taken from the tensor kernel ITSELF: whole
    #     256 x 256 tiles dumped by csg_tile_interval_sizes (same sweep, masks and accumulators as csg_action), at the
    #     places where the open-range masks and the ragged edges live: on the diagonal, next to it, the far corner, the
    #     last row/column block, and a few in between.  From them >= 10^4 RELATED pairs, half of them on rows/columns
    #     0, 1, 127, 128, 254, 255 of their tile, compared with the bit-by-bit oracle; all unrelated entries must be -1.
    rng = np.random.default_rng(cfg["seed"])
    nB = (N + 255) // 256
    tiles = [(0, 0), (0, 1), (0, nB - 1), (nB - 1, nB - 1), (nB - 2, nB - 1), (nB // 2, nB // 2), (nB // 2, nB // 2 + 1),
             (nB // 3, 2 * nB // 3), (1, nB - 2), (nB // 5, nB // 5 + 7), (nB // 7, nB - 3), (2 * nB // 3, nB - 1)]
    tiles = [(min(a, nB - 1), min(max(a, b), nB - 1)) for a, b in tiles]
    for variant in ((csg.VARIANT_TENSOR_FP4, csg.VARIANT_TENSOR) if N <= 131072 else (csg.VARIANT_TENSOR_FP4,)):
        csg.csg_set_variant(variant)
        dump = csg.csg_tile_interval_sizes(d, N, tiles).cpu().numpy()
        checked = 0
        for t, (I, J) in enumerate(tiles):
            tile = dump[t]
            rr, cc = np.nonzero(tile >= 0)
            edge = np.isin(rr, (0, 1, 127, 128, 254, 255)) | np.isin(cc, (0, 1, 127, 128, 254, 255))
            pick = np.concatenate([rng.permutation(np.nonzero(edge)[0])[:800], rng.permutation(np.nonzero(~edge)[0])[:800]])
            for k in pick:
                i, j = 256 * I + int(rr[k]), 256 * J + int(cc[k])
                assert tile[rr[k], cc[k]] == oracle.pair_interval(bits, N, i, j), (variant, I, J, i, j)
            checked += len(pick)
            ur, uc = np.nonzero(tile < 0)
            for k in rng.permutation(len(ur))[:200]:
                i, j = 256 * I + int(ur[k]), 256 * J + int(uc[k])
                assert i >= j or j >= N or oracle.pair_interval(bits, N, i, j) == -1, (variant, I, J, i, j)
        assert checked >= (10000 if dim == 2 else 3000), checked      # 4D: near-diagonal tiles hold few related pairs
    csg.csg_set_variant(csg.VARIANT_AUTO)
    # ... and the one-warp-per-pair hook on uniformly drawn pairs (mostly unrelated in 4D)
    pairs = np.sort(rng.integers(0, N, size=(2000, 2)), axis=1).astype(np.int64)
    got = csg.csg_interval_sizes(d, N, torch.from_numpy(pairs).cuda()).cpu().numpy()
    for (i, j), n in zip(pairs, got):
        assert n == oracle.pair_interval(bits, N, i, j)
    # (4) the WHOLE histogram against the oracle's stored one (Algorithm 5 over the full config, minutes of CPU, run
    #     once by tests/golden/make_config_goldens.py); the bitset hash ties the stored line to this very input
    gold = golden_histogram(cfg["name"])
    if gold is not None:
        import hashlib
        assert gold["N"] == N and csg_inputs.bits_hash(bits) == gold["bits_hash"]
        assert int(full.sum()) == gold["total"] and [int(x) for x in full[:8]] == gold["head"]
        if hashlib.sha256(np.ascontiguousarray(full, dtype="<i8").tobytes()).hexdigest() != gold["sha256"]:
            # say WHICH bins differ: recompute the oracle histogram (2D: minutes, from the coordinates)
            want = oracle.dominance2d_counts(coords, N - 2) if dim == 2 else oracle.alg5_counts(bits, N, N - 2)
            bad = np.nonzero(want != full)[0]
            raise AssertionError("histogram differs from the oracle in %d bins, first %s: got %s want %s"
                                 % (len(bad), bad[:8], full[bad[:8]], want[bad[:8]]))
        if cfg["eps"] == 1.0:
            assert float(S.item()) == oracle.action_local(dim, N, full[:4])
    # (5) else the reference histogram computed now, where Algorithm 5 finishes in reasonable time
    elif full_reference:
        want = oracle.alg5_counts(bits, N, cfg["kmax"])
        assert (counts == want).all(), (counts, want)
        if cfg["eps"] == 1.0:
            assert float(S.item()) == oracle.action_local(dim, N, want)
    if cfg["eps"] < 1.0:
        s_want, scale = oracle.action_smeared_2d(N, full, cfg["eps"])   # oracle arithmetic on the counts
        assert abs(float(S.item()) - s_want) <= 1e-12 * scale
    return counts, float(S.item())


def test_config0_plain_oracle(csg):
    cfg = csg_inputs.CONFIGS[0]
    _, bits = csg_inputs.make_causet(cfg["dim"], cfg["N"], cfg["seed"])
    want = oracle.counts_from_bits(bits, cfg["N"], cfg["kmax"])
    for variant in VARIANTS:
        got, S = run_action(csg, bits, cfg["N"], cfg["dim"], 1.0, cfg["kmax"], variant)
        assert (got == want).all() and S == oracle.action_local(2, cfg["N"], want)


def test_config1(csg):
    check_config(csg, csg_inputs.CONFIGS[1], full_reference=True)
    cfg = csg_inputs.CONFIGS[1]
    _, bits = csg_inputs.make_causet(cfg["dim"], cfg["N"], cfg["seed"])
    want = oracle.alg5_counts(bits, cfg["N"], 3)
    got, _ = run_action(csg, bits, cfg["N"], 2, 1.0, 3, 1)            # bitset variant too
    assert (got == want).all()


@pytest.mark.slow
def test_config2(csg):
    check_config(csg, csg_inputs.CONFIGS[2], full_reference=True)


@pytest.mark.slow
def test_config3_headline(csg):
    check_config(csg, csg_inputs.CONFIGS[3], full_reference=True)


@pytest.mark.slow
def test_config4_smeared(csg):
    """All 262143 bins and S against the oracle's stored histogram (tests/golden/config_histograms.txt, written from
    oracle/dominance2d.c); this is the configuration that runs the throttled instantiation of the fp4 kernel."""
    assert golden_histogram(csg_inputs.CONFIGS[4]["name"]) is not None
    check_config(csg, csg_inputs.CONFIGS[4], full_reference=False)


# --------------------------------------------------------------------------- the tensor kernel's own n_ij, pair by pair
@pytest.mark.parametrize("variant", [2, 3])
@pytest.mark.parametrize("dim,N,seed", [(2, 700, 1), (4, 1300, 2), (2, 2049, 3)])
def test_tile_dump_equals_oracle_pair_by_pair(csg, variant, dim, N, seed):
    """csg_tile_interval_sizes: every entry of every tile against the definition (U @ U on the expanded matrix)."""
    _, bits = csg_inputs.make_causet(dim, N, seed)
    U = np.triu(oracle.expand(bits, N), 1).astype(np.int64)
    want = np.where(U == 1, U @ U, -1)
    nB = (N + 255) // 256
    tiles = [(I, J) for I in range(nB) for J in range(I, nB)]
    csg.csg_set_variant(variant)
    dump = csg.csg_tile_interval_sizes(csg.to_device(bits), N, tiles).cpu().numpy()
    csg.csg_set_variant(csg.VARIANT_AUTO)
    padded = np.full((256 * nB, 256 * nB), -1, dtype=np.int64)
    padded[:N, :N] = want
    for t, (I, J) in enumerate(tiles):
        assert (dump[t] == padded[256 * I:256 * I + 256, 256 * J:256 * J + 256]).all(), (I, J)


# --------------------------------------------------------------------------- the throttled instantiation under a live oracle
@pytest.mark.parametrize("dim,N,kmax", [(2, 16384, 16382), (4, 9001, 3), (2, 5000, 4998)])
def test_throttled_instantiation_equals_oracle(csg, dim, N, kmax):
    """CSG_THROTTLE_ON selects the instantiation of the fp4 kernel that BASELINE.json configs[4] runs (TMA threads wait
    on the finished-tile counter) at sizes where Algorithm 5 finishes in seconds; results must not depend on it."""
    _, bits = csg_inputs.make_causet(dim, N, 31 + N)
    want = oracle.alg5_counts(bits, N, kmax)
    d = csg.to_device(bits)
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    try:
        for mode in (csg.THROTTLE_ON, csg.THROTTLE_OFF, csg.THROTTLE_ON):
            csg.csg_set_throttle(mode)
            for _ in range(3):
                c, S = csg.csg_action(d, N, dim, 1.0, kmax)
                torch.cuda.synchronize()
                assert (c.cpu().numpy() == want).all(), mode
                assert float(S.item()) == oracle.action_local(dim, N, want)
    finally:
        csg.csg_set_throttle(csg.THROTTLE_AUTO)
        csg.csg_set_variant(csg.VARIANT_AUTO)


# --------------------------------------------------------------------------- cached state: sizes, shards, streams, graphs
def test_alternating_sizes_shards_and_streams_without_sync(csg):
    """After one warm-up call per (N, shard) csg_action / csg_action_partial only enqueue: alternating two sizes and
    three shards on two streams never synchronises (the call returns while its stream is still busy) and every
    result is bit-exact."""
    csg.csg_set_variant(csg.VARIANT_AUTO)
    sizes = [(4, 2600), (2, 1900)]
    sets = {N: csg_inputs.make_causet(dim, N, 50 + N)[1] for dim, N in sizes}
    want = {N: oracle.alg5_counts(sets[N], N, 3) for _, N in sizes}
    dev = {N: csg.to_device(sets[N]) for _, N in sizes}
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for dim, N in sizes:                                              # warm-up: builds the cached tile schedules
        csg.csg_action(dev[N], N, dim, 1.0, 3)
        for s in range(3):
            csg.csg_action_partial(dev[N], N, 3, s, 3)
    torch.cuda.synchronize()
    results = []
    busy_seen = 0
    for it in range(12):
        dim, N = sizes[it % 2]
        st = streams[(it // 2) % 2]
        with torch.cuda.stream(st):
            torch.cuda._sleep(40_000_000)                             # ~20 ms of busy stream ahead of the call
            c, S = csg.csg_action(dev[N], N, dim, 1.0, 3, stream=st)
            parts = [csg.csg_action_partial(dev[N], N, 3, s, 3, stream=st) for s in range(3)]
            busy_seen += not st.query()                               # had the call synchronised, the stream would be idle
        results.append((N, dim, c, S, parts))
    torch.cuda.synchronize()
    assert busy_seen >= 10, busy_seen
    for N, dim, c, S, parts in results:
        assert (c.cpu().numpy() == want[N]).all()
        assert (sum(parts).cpu().numpy() == want[N]).all()
        assert float(S.item()) == oracle.action_local(dim, N, want[N])


def test_graph_survives_other_sizes(csg):
    """A captured csg_action keeps working after calls with other sizes (cached tile lists are never freed or
    overwritten before csg_shutdown)."""
    csg.csg_set_variant(csg.VARIANT_AUTO)
    N1, N2, N3 = 3000, 1700, 5200
    b1, b2, b3 = (csg_inputs.make_causet(4, N, 60 + N)[1] for N in (N1, N2, N3))
    d1, d2, d3 = csg.to_device(b1), csg.to_device(b2), csg.to_device(b3)
    c1 = torch.zeros(4, dtype=torch.int64, device="cuda")
    S1 = torch.zeros(1, dtype=torch.float64, device="cuda")
    csg.csg_action(d1, N1, 4, 1.0, 3, c1, S1)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        csg.csg_action(d1, N1, 4, 1.0, 3, c1, S1)
    want1 = oracle.alg5_counts(b1, N1, 3)
    for other_d, other_N, other_b in ((d2, N2, b2), (d3, N3, b3), (d2, N2, b2)):
        c, _ = csg.csg_action(other_d, other_N, 4, 1.0, 3)
        for s in range(2):
            csg.csg_action_partial(other_d, other_N, 3, s, 2)
        torch.cuda.synchronize()
        assert (c.cpu().numpy() == oracle.alg5_counts(other_b, other_N, 3)).all()
        c1.fill_(-1)
        graph.replay()
        torch.cuda.synchronize()
        assert (c1.cpu().numpy() == want1).all()
        assert float(S1.item()) == oracle.action_local(4, N1, want1)


def test_fused_small_sets_on_streams_and_in_graphs(csg):
    """N <= 1024 (bitset variant): eager calls take the fused single launch (one kernel per action, per-stream
    workspace), captured calls the three-node path; both bit-exact, interleaved on two streams, local and smeared."""
    csg.csg_set_variant(csg.VARIANT_AUTO)
    cases = [(2, 1024, 1.0, 3), (4, 700, 1.0, 3), (2, 513, 0.1, 511), (2, 64, 1.0, 62), (2, 3, 1.0, 2)]
    data = []
    for dim, N, eps, kmax in cases:
        _, bits = csg_inputs.make_causet(dim, N, 800 + N)
        want = oracle.counts_from_bits(bits, N, kmax)
        data.append((dim, N, eps, kmax, csg.to_device(bits), want))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    l0 = csg.csg_launch_count()
    out = []
    for rep in range(6):
        for k, (dim, N, eps, kmax, d, want) in enumerate(data):
            st = streams[(rep + k) % 2]
            with torch.cuda.stream(st):
                out.append((k, csg.csg_action(d, N, dim, eps, kmax, stream=st)))
    torch.cuda.synchronize()
    assert csg.csg_launch_count() - l0 == 6 * len(cases)              # ONE kernel per action
    for k, (c, S) in out:
        dim, N, eps, kmax, d, want = data[k]
        assert (c.cpu().numpy() == want).all(), (N, eps)
        if eps == 1.0:
            assert float(S.item()) == oracle.action_local(dim, N, np.concatenate([want, np.zeros(4, np.int64)]))
        else:
            s_want, scale = oracle.action_smeared_2d(N, want, eps)
            assert abs(float(S.item()) - s_want) <= 1e-12 * scale
    # same S bits from the fused launch, the three-node path (inside a graph) and the batch call
    dim, N, eps, kmax, d, want = data[2]
    c_e, S_e = csg.csg_action(d, N, dim, eps, kmax)
    c_g = torch.zeros(kmax + 1, dtype=torch.int64, device="cuda")
    S_g = torch.zeros(1, dtype=torch.float64, device="cuda")
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        csg.csg_action(d, N, dim, eps, kmax, c_g, S_g)
    graph.replay()
    c_b, S_b = csg.csg_action_batch(d, N, 1, dim, eps, kmax)
    torch.cuda.synchronize()
    assert torch.equal(c_e, c_g) and torch.equal(c_e, c_b[0])
    assert float(S_e.item()) == float(S_g.item()) == float(S_b[0].item())


def test_measure_peak_runs(csg):
    for what in (csg.PEAK_MMA_MXF4, csg.PEAK_MMA_I8, csg.PEAK_ALU_MIX, csg.PEAK_ALU_POPC, csg.PEAK_ALU_LOP3):
        ms, units = csg.csg_measure_peak(what, 2000)
        assert ms > 0 and units > 0
    ms, units = csg.csg_measure_peak(csg.PEAK_MMA_MXF4, 20000)
    rate = units / (ms * 1e-3)                                        # MAC/s over the device
    assert 1.5e15 < rate < 6e15, rate                                 # nominal dense fp4: 4.5e15 MAC/s


@pytest.mark.parametrize("N,dim", [(1000, 2), (3000, 4)])
def test_csg_action_is_cuda_graph_capturable(csg, N, dim):
    """After one warm-up call (which builds the cached tile schedule) csg_action only enqueues stream-ordered work, so a
    launch-bound loop over small causal sets can be captured in a CUDA graph and replayed."""
    csg.csg_set_variant(csg.VARIANT_AUTO)
    sets = [csg_inputs.make_causet(dim, N, 900 + b)[1] for b in range(4)]
    d = [csg.to_device(b) for b in sets]
    counts = [torch.zeros(4, dtype=torch.int64, device="cuda") for _ in sets]
    S = [torch.zeros(1, dtype=torch.float64, device="cuda") for _ in sets]
    csg.csg_action(d[0], N, dim, 1.0, 3, counts[0], S[0])            # warm-up outside the capture
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        for b in range(4):
            csg.csg_action(d[b], N, dim, 1.0, 3, counts[b], S[b])
    for c in counts:
        c.fill_(-1)
    graph.replay()
    torch.cuda.synchronize()
    for b in range(4):
        want = reference_counts(sets[b], N, 3)
        assert (counts[b].cpu().numpy() == want).all()
        assert float(S[b].item()) == oracle.action_local(dim, N, want)
