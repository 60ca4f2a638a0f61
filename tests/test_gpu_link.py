"""Parity of the linking kernel (csg_link, through the C ABI) with the linking oracle, bit for bit, and of the
coordinates-in / action-out call with the action oracle."""
import math

import numpy as np
import pytest

import csg_inputs
import oracle

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

M2, M4, DS = 0, 1, 2


@pytest.fixture(scope="module")
def csg():
    import paper_1709_03013_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    if m._build.needs_build():
        m.build()
    m.load()
    m.csg_set_variant(m.VARIANT_AUTO)
    return m


def coords_for(geom, N, seed):
    if geom == DS:
        return csg_inputs.sprinkle_de_sitter(N, seed)
    return csg_inputs.sprinkle(4 if geom == M4 else 2, N, seed)


def gpu_link(csg, coords, geom, poison=True):
    N = coords.shape[0]
    d = torch.from_numpy(coords).cuda()
    out = torch.full((N, csg.csg_row_stride_words(N)), -1 if poison else 0, dtype=torch.int64, device="cuda")
    csg.csg_link(d, N, geom, out)
    torch.cuda.synchronize()
    return out.cpu().numpy().view(np.uint64)


@pytest.mark.parametrize("geom", [M2, M4, DS])
@pytest.mark.parametrize("N", [1, 2, 3, 63, 255, 256, 257, 511, 513, 700, 1500, 3000])
def test_link_matches_oracle_bit_for_bit(csg, geom, N):
    """Every word, padding included (the output buffer is pre-filled with ones)."""
    coords = coords_for(geom, N, 100 + N)
    want = csg_inputs.pack_dense(np.triu(oracle.link(geom, coords), 1))
    got = gpu_link(csg, coords, geom)
    assert got.shape == want.shape
    assert (got == want).all(), np.argwhere(got != want)[:5]


@pytest.mark.parametrize("geom", [M2, M4, DS])
def test_link_degenerate_inputs(csg, geom):
    """Equal times / coincident events (no relation under strict inequalities) and a total order."""
    N = 600
    dim = 4 if geom == M4 else 2
    same = np.zeros((N, dim))
    assert gpu_link(csg, same, geom).sum() == 0
    t = np.linspace(0.0, 1.0, N) if geom != DS else np.linspace(-0.5, 0.5, N)
    chain = np.zeros((N, dim))
    chain[:, 0] = t
    if geom == M2:
        chain[:, 1] = t
    want = csg_inputs.pack_dense(np.triu(np.ones((N, N)), 1))
    assert (gpu_link(csg, chain, geom) == want).all()


@pytest.mark.parametrize("geom,N,eps", [(M2, 1800, 1.0), (M4, 2500, 1.0), (DS, 2200, 2.0 ** -6), (M2, 900, 0.1)])
def test_coordinates_in_action_out(csg, geom, N, eps):
    coords = coords_for(geom, N, 7 + N)
    bits = csg_inputs.pack_dense(np.triu(oracle.link(geom, coords), 1))
    dim = 4 if geom == M4 else 2
    kmax = 3 if eps == 1.0 else N - 2
    want = oracle.alg5_counts(bits, N, kmax)
    counts, S = csg.csg_causet_action_host(coords, N, geom, eps, kmax)
    assert (counts == want).all()
    if eps == 1.0:
        assert S == oracle.action_local(dim, N, want)
    else:
        s_want, scale = oracle.action_smeared_2d(N, want, eps)
        assert abs(S - s_want) <= 1e-12 * scale
    # device-resident composition gives the same
    d_bits = csg.csg_link(torch.from_numpy(coords).cuda(), N, geom)
    c2, S2 = csg.csg_action(d_bits, N, dim, eps, kmax)
    torch.cuda.synchronize()
    assert (c2.cpu().numpy() == want).all() and float(S2.item()) == S


def test_link_error_codes(csg):
    d = torch.zeros(64, dtype=torch.float64, device="cuda")
    out = torch.zeros(64, dtype=torch.int64, device="cuda")
    lib = csg.load()
    for args, code in [((None, 8, 0, out.data_ptr(), None), -1), ((d.data_ptr(), 0, 0, out.data_ptr(), None), -2),
                       ((d.data_ptr(), 8, 3, out.data_ptr(), None), -11), ((d.data_ptr(), 8, 0, out.data_ptr() + 8, None), -3)]:
        with pytest.raises(csg.CsgError) as e:
            csg._check(lib.csg_link(*args))
        assert e.value.code == code


# --------------------------------------------------------------------------- full-size configurations
def check_full_size(csg, geom, N, seed, bits=None):
    """At sizes where the N x N byte oracle cannot run: (1) the linking oracle on a random sub-causal-set (a relation
    depends on its two elements only), (2) the whole matrix against the host generator's, which the CPU pins
    tie to the oracle."""
    coords = coords_for(geom, N, seed)
    d_bits = csg.csg_link(torch.from_numpy(coords).cuda(), N, geom)
    torch.cuda.synchronize()
    rng = np.random.default_rng(seed)
    idx = np.sort(rng.choice(N, size=1500, replace=False))
    idx[:40] = np.arange(40)                       # keep some near-diagonal pairs and the ragged end
    idx[-40:] = np.arange(N - 40, N)
    idx = np.unique(idx)
    B = oracle.link(geom, coords[idx])
    rows = d_bits[torch.from_numpy(idx).cuda()].cpu().numpy().view(np.uint64)
    got = ((rows[:, idx // 64] >> (idx % 64).astype(np.uint64)) & np.uint64(1)).astype(np.uint8)
    assert (got == B).all()
    if bits is None:
        bits = csg_inputs.relations_de_sitter(coords) if geom == DS else csg_inputs.relations_from_coords(coords)
    same = bool((d_bits.cpu().numpy().view(np.uint64) == bits).all())
    assert same
    return coords, d_bits


def test_link_config1(csg):
    cfg = csg_inputs.CONFIGS[1]
    check_full_size(csg, M2, cfg["N"], cfg["seed"])


@pytest.mark.slow
def test_link_config3_headline(csg):
    cfg = csg_inputs.CONFIGS[3]
    coords, d_bits = check_full_size(csg, M4, cfg["N"], cfg["seed"])
    counts, S = csg.csg_action(d_bits, cfg["N"], 4, 1.0, 3)       # linked on the device, then the action
    torch.cuda.synchronize()
    c_host, S_host = csg.csg_causet_action_host(coords, cfg["N"], M4, 1.0, 3)
    assert (counts.cpu().numpy() == c_host).all() and float(S.item()) == S_host


@pytest.mark.slow
def test_link_config4(csg):
    cfg = csg_inputs.CONFIGS[4]
    check_full_size(csg, M2, cfg["N"], cfg["seed"])


@pytest.mark.slow
def test_de_sitter_mean_action_approaches_einstein_hilbert(csg):
    """The paper's own workload and its only printed physics value (Fig. 4, Eq. 10): the
    (1+1) de Sitter slab eta0 = 0.5, eps = 2^-6, mean over ten graphs converging to S_EH = 4 pi tan(eta0) = 6.865
    for N >~ 2^14.  Soft check (the figure's values are not printed): the mean of ten graphs at N = 2^15 is within
    four standard errors + 15 % of S_EH."""
    N, eps, eta0 = 1 << 15, 2.0 ** -6, 0.5
    S = []
    for g in range(10):
        coords = csg_inputs.sprinkle_de_sitter(N, 31000 + g, eta0)
        _, s = csg.csg_causet_action_host(coords, N, DS, eps, N - 2)
        S.append(s)
    S = np.array(S)
    s_eh = 4 * math.pi * math.tan(eta0)
    sem = S.std(ddof=1) / math.sqrt(len(S))
    print("de Sitter N=%d: mean S = %.3f +- %.3f (S_EH = %.3f), sigma = %.3f" % (N, S.mean(), sem, s_eh, S.std(ddof=1)))
    assert abs(S.mean() - s_eh) <= 4 * sem + 0.15 * s_eh


# --------------------------------------------------------------------------- the single-precision filter of the 4D kernel
def _sorted_by_time(c):
    return np.ascontiguousarray(c[np.argsort(c[:, 0], kind="stable")])


@pytest.mark.parametrize("offset,scale", [(0.0, 1.0), (1000.0, 1.0), (-3.0e6, 1.0), (0.0, 1.0e-12), (0.0, 1.0e9),
                                          (0.0, 1.0e17), (7.0, 3.0e-5)])
def test_link_4d_filter_near_the_light_cone(csg, offset, scale):
    """Pairs exactly on the cone, one ulp inside and one ulp outside it, among ordinary events; every coordinate
    shifted and scaled so that the certainty bound of the single-precision test is tiny, huge or switched off.  The
    kernel must take the double-precision decision for every pair: word for word equal to the linking oracle."""
    rng = np.random.default_rng(int(abs(offset)) + 17)
    base = csg_inputs.sprinkle(4, 700, 4242)
    extra = []
    for k in range(120):
        a = base[rng.integers(0, 700)].copy()
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        r = rng.uniform(0.01, 0.3)
        b = a.copy()
        b[1:] += r * d
        dist = math.sqrt(float(((b[1:] - a[1:]) ** 2).sum()))
        dt = [dist, np.nextafter(dist, 2.0), np.nextafter(dist, 0.0), dist * (1 + 3e-8), dist * (1 - 3e-8)][k % 5]
        b[0] = a[0] + dt
        extra.append(b)
    # pythagorean displacements: exactly on the cone in exact arithmetic
    for q in range(1, 9):
        extra.append(np.array([0.125 + 5.0 / 64 * q / 8, 3.0 / 64 * q / 8, 4.0 / 64 * q / 8, 0.0]))
    extra.append(np.array([0.125, 0.0, 0.0, 0.0]))
    coords = _sorted_by_time(np.vstack([base, np.array(extra)]) * scale + offset * scale)
    want = csg_inputs.pack_dense(np.triu(oracle.link(M4, coords), 1))
    got = gpu_link(csg, coords, M4)
    assert (got == want).all(), np.argwhere(got != want)[:5]


def test_link_4d_filter_nan_and_inf(csg):
    """NaN and infinite coordinates never relate anything under the strict double-precision tests; the filter must not
    decide them either."""
    coords = _sorted_by_time(csg_inputs.sprinkle(4, 520, 99))
    coords[100, 1] = np.nan
    coords[300, 0] = np.inf
    coords[301, 2] = -np.inf
    with np.errstate(invalid="ignore"):
        want = csg_inputs.pack_dense(np.triu(oracle.link(M4, coords), 1))
    got = gpu_link(csg, coords, M4)
    assert (got == want).all(), np.argwhere(got != want)[:5]
