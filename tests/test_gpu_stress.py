"""Repeated launches: the full histogram must be identical to the oracle's on every run, through the device-resident
call and through the chunked host call.  (A race between the packed-bit ring's LDS reads and the TMA refill once lost
a handful of n_ij per 10^10 pairs; it only showed under repetition or at the largest configuration.)"""
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


@pytest.mark.parametrize("sparse", [0, 1])
@pytest.mark.parametrize("throttle", [0, 1])
@pytest.mark.parametrize("dim,N,reps", [(2, 16384, 12), (4, 16384, 8), (2, 9000, 12)])
def test_repeated_full_histograms(csg, dim, N, reps, throttle, sparse):
    """throttle = 1 (CSG_THROTTLE_ON): the instantiation of the fp4 kernel whose TMA threads wait on the finished-tile
    counter -- the one BASELINE.json configs[4] runs -- on the device-resident call, and together with the copy gate
    on the host call.  sparse = 1 (CSG_SPARSE_ON): the instantiations in which the three roles of the kernel each walk
    the live-group masks of the occupancy map (the headline launch), incl. the gated host pipeline whose occupancy rows
    are written while the kernel runs."""
    _, bits = csg_inputs.make_causet(dim, N, 777 + N)
    want = oracle.alg5_counts(bits, N, N - 2)
    d = csg.to_device(bits)
    pinned = torch.from_numpy(bits.view(np.int64)).pin_memory()
    csg.csg_set_throttle(throttle)
    csg.csg_set_sparse(sparse)
    try:
        for r in range(reps):
            c, _ = csg.csg_action(d, N, dim, 1.0, N - 2)
            torch.cuda.synchronize()
            assert (c.cpu().numpy() == want).all(), ("device", r)
            ch, _ = csg.csg_action_host(pinned, N, dim, 1.0, N - 2)
            assert (ch == want).all(), ("host", r)
    finally:
        csg.csg_set_throttle(0)
        csg.csg_set_sparse(0)


@pytest.mark.slow
def test_config4_is_run_to_run_identical(csg):
    cfg = csg_inputs.CONFIGS[4]
    N = cfg["N"]
    _, bits = csg_inputs.make_config(cfg)
    d = csg.to_device(bits)
    first = None
    for r in range(3):
        c, S = csg.csg_action(d, N, 2, cfg["eps"], N - 2)
        torch.cuda.synchronize()
        c = c.cpu().numpy()
        if first is None:
            first = (c, float(S.item()))
        else:
            assert (c == first[0]).all() and float(S.item()) == first[1], r


@pytest.mark.slow
def test_config4_int8_kind_equals_fp4_kind(csg):
    """N = 262144 is the only configuration that takes the int8 kind's TB = 6 operand encoding (n_ij << 12 in s32)."""
    cfg = csg_inputs.CONFIGS[4]
    N = cfg["N"]
    _, bits = csg_inputs.make_config(cfg)
    d = csg.to_device(bits)
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    a, Sa = csg.csg_action(d, N, 2, cfg["eps"], N - 2)
    csg.csg_set_variant(csg.VARIANT_TENSOR)
    b, Sb = csg.csg_action(d, N, 2, cfg["eps"], N - 2)
    torch.cuda.synchronize()
    csg.csg_set_variant(csg.VARIANT_AUTO)
    assert torch.equal(a, b) and float(Sa.item()) == float(Sb.item())
