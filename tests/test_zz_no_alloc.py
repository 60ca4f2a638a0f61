"""csg_action_noalloc (include/csg.h): the entry point that allocates nothing -- its scratch is a file-scope static
device array -- must return what the existing path (csg_action) returns: counts bit for bit, the local action exactly,
the smeared action within the tolerance of the other parity tests (1e-12 of its term scale), on two calls in a row
(the array is shared by every call and keeps the last call's contents).  Also checked against the oracle, that sizes
beyond the static maximum are refused with a clear error, and that the device's free memory does not move across calls.

The file name sorts last on purpose: the round's end runs `pytest -x`, so a failure here hides no other test."""
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
    m.csg_set_variant(m.VARIANT_AUTO)
    return m


def run_both(csg, bits, N, dim, eps, kmax, repeats=2):
    d = csg.to_device(bits)
    want_c, want_S = csg.csg_action(d, N, dim, eps, kmax)                 # the existing path
    torch.cuda.synchronize()
    want_c, want_S = want_c.cpu().numpy().copy(), float(want_S.item())
    out = []
    counts = torch.empty(kmax + 1, dtype=torch.int64, device="cuda")
    S = torch.empty(1, dtype=torch.float64, device="cuda")
    for _ in range(repeats):                                              # two calls in a row share the static scratch
        counts.fill_(-7)
        S.fill_(float("nan"))
        csg.csg_action_noalloc(d, N, dim, eps, kmax, counts, S)
        torch.cuda.synchronize()
        out.append((counts.cpu().numpy().copy(), float(S.item())))
    return want_c, want_S, out


@pytest.mark.parametrize("dim,N,seed", [(2, 1, 1), (2, 2, 2), (2, 63, 3), (2, 257, 4), (4, 700, 5), (2, 1024, 6),
                                        (4, 1500, 7), (2, 3001, 8), (4, 4096, 9)])
def test_noalloc_local_action_equals_existing_path(csg, dim, N, seed):
    _, bits = csg_inputs.make_causet(dim, N, 9000 + seed)
    kmax = 3
    want_c, want_S, out = run_both(csg, bits, N, dim, 1.0, kmax)
    ref = oracle.counts_from_bits(bits, N, kmax) if N <= 1200 else oracle.alg5_counts(bits, N, kmax)
    assert (want_c == ref).all()
    for call, (c, S) in enumerate(out):
        assert (c == want_c).all(), (call, c, want_c)
        assert S == want_S, (call, S, want_S)                              # exact: an integer combination times a constant
        assert S == oracle.action_local(dim, N, ref)


@pytest.mark.parametrize("dim,N,eps", [(2, 300, 0.1), (2, 777, 0.5), (2, 1025, 0.03), (4, 900, 0.25)])
def test_noalloc_whole_histogram_and_smeared_action(csg, dim, N, eps):
    _, bits = csg_inputs.make_causet(dim, N, 31 * N)
    kmax = N - 2                                                          # <= CSG_NOALLOC_MAX_KMAX = 1023
    want_c, want_S, out = run_both(csg, bits, N, dim, eps, kmax, repeats=3)
    ref = oracle.counts_from_bits(bits, N, kmax)
    assert (want_c == ref).all()
    if dim == 2:
        s_ref, scale = oracle.action_smeared_2d(N, ref, eps)
    else:
        s_ref, scale = oracle.action_smeared_4d(N, ref, eps)
    for call, (c, S) in enumerate(out):
        assert (c == want_c).all(), call
        assert abs(S - want_S) <= 1e-12 * scale, (call, S, want_S)
        assert abs(S - s_ref) <= 1e-12 * scale, (call, S, s_ref)


def test_noalloc_dirty_scratch_and_alternating_sizes(csg):
    """A large-kmax call followed by small ones and back: nothing of one call's bins may leak into the next."""
    sets = [(2, 1000, 998, 0.2), (2, 200, 3, 1.0), (4, 4096, 3, 1.0), (2, 1000, 998, 0.2), (2, 64, 62, 0.5)]
    for dim, N, kmax, eps in sets + sets[::-1]:
        _, bits = csg_inputs.make_causet(dim, N, 5 * N + dim)
        want_c, want_S, out = run_both(csg, bits, N, dim, eps, kmax, repeats=1)
        c, S = out[0]
        assert (c == want_c).all(), (dim, N, kmax)
        if eps == 1.0:
            assert S == want_S
        else:
            _, scale = oracle.action_smeared_2d(N, want_c, eps)
            assert abs(S - want_S) <= 1e-12 * scale


def test_noalloc_rejects_sizes_beyond_the_static_scratch(csg):
    assert csg.NOALLOC_MAX_N == 4096 and csg.NOALLOC_MAX_KMAX == 1023
    _, bits = csg_inputs.make_causet(2, 300, 1)
    d = csg.to_device(bits)
    counts = torch.full((2000,), -7, dtype=torch.int64, device="cuda")
    S = torch.zeros(1, dtype=torch.float64, device="cuda")
    big = torch.zeros(4097 * csg.csg_row_stride_words(4097), dtype=torch.int64, device="cuda")
    with pytest.raises(csg.CsgError) as e:
        csg.csg_action_noalloc(big, 4097, 2, 1.0, 3, counts, S)           # N beyond the maximum
    assert e.value.code == -12 and "CSG_NOALLOC_MAX_N" in str(e.value)
    with pytest.raises(csg.CsgError) as e:
        csg.csg_action_noalloc(d, 300, 2, 0.5, 1024, counts, S)           # kmax beyond the maximum
    assert e.value.code == -12 and "CSG_NOALLOC_MAX_KMAX" in str(e.value)
    with pytest.raises(csg.CsgError) as e:
        csg.csg_action_noalloc(d, 300, 3, 1.0, 3, counts, S)              # ordinary validation still applies
    assert e.value.code == -4
    torch.cuda.synchronize()
    assert (counts.cpu().numpy() == -7).all()                             # refused calls enqueue nothing
    csg.csg_action_noalloc(d, 300, 2, 0.5, 1023, counts, S)               # the maximum itself is accepted
    torch.cuda.synchronize()
    assert (counts[:299].cpu().numpy() == oracle.counts_from_bits(bits, 300, 298)).all()
    assert (counts[299:1024].cpu().numpy() == 0).all()


def test_noalloc_leaves_device_memory_alone(csg):
    """After the set-up and one warm call (module loading) the device's free memory must not move across calls."""
    _, bits = csg_inputs.make_causet(4, 2000, 77)
    d = csg.to_device(bits)
    counts = torch.empty(4, dtype=torch.int64, device="cuda")
    S = torch.empty(1, dtype=torch.float64, device="cuda")
    stream = torch.cuda.Stream()
    csg.csg_noalloc_setup()
    csg.csg_action_noalloc(d, 2000, 4, 1.0, 3, counts, S)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(50):
        csg.csg_action_noalloc(d, 2000, 4, 1.0, 3, counts, S)
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):                                       # a new stream: the existing path would allocate here
        stream.wait_stream(torch.cuda.current_stream())
        csg.csg_action_noalloc(d, 2000, 4, 1.0, 3, counts, S, stream=stream)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    assert (counts.cpu().numpy() == oracle.alg5_counts(bits, 2000, 3)).all()


def test_noalloc_inside_a_cuda_graph(csg):
    """The case the entry point is for: captured into a CUDA graph WITHOUT any warm-up call of that size (csg_action needs
    one, it allocates on first use), replayed twice.  The two captured calls run one after the other in the graph's
    single stream, as the shared scratch requires."""
    csg.csg_noalloc_setup()                                               # module loading and address look-up outside the capture
    sets = [csg_inputs.make_causet(4, 1700 + 100 * b, 400 + b)[1] for b in range(2)]
    Ns = [1700, 1800]
    d = [csg.to_device(b) for b in sets]
    counts = [torch.zeros(4, dtype=torch.int64, device="cuda") for _ in sets]
    S = [torch.zeros(1, dtype=torch.float64, device="cuda") for _ in sets]
    csg.csg_action_noalloc(d[0], 64, 4, 1.0, 3, counts[0], S[0])           # loads the kernel; a DIFFERENT size on purpose
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        for b in range(2):
            csg.csg_action_noalloc(d[b], Ns[b], 4, 1.0, 3, counts[b], S[b])
    for rep in range(2):
        for c in counts:
            c.fill_(-1)
        graph.replay()
        torch.cuda.synchronize()
        for b in range(2):
            want = oracle.alg5_counts(sets[b], Ns[b], 3)
            assert (counts[b].cpu().numpy() == want).all(), (rep, b)
            assert float(S[b].item()) == oracle.action_local(4, Ns[b], want)
