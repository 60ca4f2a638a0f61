"""Pins of the linking oracle (oracle/link_oracle.c) against what the paper and the mathematics fix --
none of them re-types the oracle's formula.  CPU only."""
import math

import numpy as np
import pytest

import csg_inputs
import oracle

M2, M4, DS = oracle.GEOM_MINKOWSKI_2D, oracle.GEOM_MINKOWSKI_4D, oracle.GEOM_DESITTER_2D


def _inversions(a):
    """Number of pairs p<q with a[p] > a[q], by merge sort (pure Python, O(n log n))."""
    a = list(a)
    if len(a) < 2:
        return 0, a
    mid = len(a) // 2
    il, left = _inversions(a[:mid])
    ir, right = _inversions(a[mid:])
    out, inv, p, q = [], il + ir, 0, 0
    while p < len(left) and q < len(right):
        if left[p] <= right[q]:
            out.append(left[p]); p += 1
        else:
            out.append(right[q]); q += 1; inv += len(left) - p
    out += left[p:] + right[q:]
    return inv, out


@pytest.mark.parametrize("N,seed", [(2, 1), (3, 2), (257, 3), (1500, 4)])
def test_2d_relation_count_is_non_inversions(N, seed):
    """A 2D order from (u, v): #relations = C(N,2) - inversions of the v-ranks read in u-order.
    Also pins the time sort: a relation i<j stored against the index order would go missing."""
    coords = csg_inputs.sprinkle(2, N, seed)
    B = oracle.link(M2, coords)
    v_in_u_order = coords[np.argsort(coords[:, 0]), 1]
    inv, _ = _inversions(v_in_u_order)
    assert int(np.triu(B, 1).sum()) == N * (N - 1) // 2 - inv


def test_4d_hand_events_on_inside_outside_the_cone():
    """dt^2 > dx^2+dy^2+dz^2 strictly: inside related, on the cone (null) and outside unrelated, equal times
    unrelated.  Rows sorted by t."""
    ev = np.array([[0.0, 0.0, 0.0, 0.0],
                   [1.0, 0.5, 0.0, 0.0],     # inside the cone of event 0
                   [1.0, 1.0, 0.0, 0.0],     # on the cone of event 0 (null): unrelated
                   [1.0, 0.6, 0.6, 0.6],     # 1.08 > 1: outside
                   [2.0, 1.0, 1.0, 1.0]])    # 4 > 3: inside the cone of event 0; from event 1: 1 > 0.25+1+1? no
    B = oracle.link(M4, ev)
    want = np.zeros((5, 5), np.uint8)
    for i, j in [(0, 1), (0, 4), (3, 4)]:    # (3,4): dt=1, d^2 = .16*3 = .48 < 1
        want[i, j] = want[j, i] = 1
    # (1,4): dt=1, d^2 = .25+1+1 > 1 no; (2,4): dt=1, d^2 = 0+1+1 no; (1,2),(1,3),(2,3): equal times
    assert (B == want).all()


def test_de_sitter_hand_events_wrap_around():
    """pi - |pi - |dtheta|| < |deta|.  The angle difference wraps around 2 pi."""
    ev = np.array([[-0.4, 0.1],
                   [0.3, 6.2],     # |dtheta| = 6.1 -> wrapped 2pi-6.1 = 0.183 < 0.7: related to event 0
                   [0.3, 1.0],     # 0.9 > 0.7: unrelated to event 0; equal eta with event 1: unrelated
                   [0.45, 0.9]])   # from 0: .8 < .85 related; from 1: wrapped .983 > .15 no; from 2: .1 < .15 related
    B = oracle.link(DS, ev)
    want = np.zeros((4, 4), np.uint8)
    for i, j in [(0, 1), (0, 3), (2, 3)]:
        want[i, j] = want[j, i] = 1
    assert (B == want).all()


def test_chain_and_antichain():
    N = 40
    t = np.arange(N, dtype=np.float64)
    chain = np.stack([t, 0 * t, 0 * t, 0 * t], 1)            # events on a timelike line: total order
    assert (oracle.link(M4, chain) == 1 - np.eye(N, dtype=np.uint8)).all()
    simultaneous = np.stack([0 * t, t, 0 * t, 0 * t], 1)      # equal times: antichain
    assert oracle.link(M4, simultaneous).sum() == 0
    diag = np.stack([t, t], 1)                                 # u = v increasing: chain in light-cone coords
    assert (oracle.link(M2, diag) == 1 - np.eye(N, dtype=np.uint8)).all()
    anti = np.stack([t, -t], 1)                                # u up, v down: antichain
    assert oracle.link(M2, anti).sum() == 0


@pytest.mark.parametrize("geom", [M2, M4, DS])
def test_result_is_a_symmetric_irreflexive_transitive_order(geom):
    N = 500
    coords = csg_inputs.sprinkle_de_sitter(N, 9) if geom == DS else csg_inputs.sprinkle(4 if geom == M4 else 2, N, 9)
    B = oracle.link(geom, coords)
    assert (B == B.T).all() and np.trace(B) == 0
    U = np.triu(B, 1).astype(np.int64)
    two_step = (U @ U) > 0                                    # i < k < j with i~k and k~j
    assert (U[two_step] == 1).all()                           # causal orders are transitive


def test_4d_ordering_fraction_is_one_tenth():
    """Alexandrov interval of d-dimensional Minkowski space: E[#relations]/C(N,2) =
    Gamma(d+1) Gamma(d/2) / (2 Gamma(3d/2)); d=2: 1/2, d=4: 1/10 (Myrheim-Meyer)."""
    assert math.gamma(5) * math.gamma(2) / (2 * math.gamma(6)) == pytest.approx(0.1)
    N, fr = 300, []
    for seed in range(40):
        B = oracle.link(M4, csg_inputs.sprinkle(4, N, 1000 + seed))
        fr.append(np.triu(B, 1).sum() / (N * (N - 1) / 2))
    fr = np.array(fr)
    assert abs(fr.mean() - 0.1) <= 4 * fr.std(ddof=1) / math.sqrt(len(fr))
    assert 0.001 < fr.std(ddof=1) < 0.02


def test_de_sitter_ordering_fraction_matches_quadrature():
    """theta uniform on the circle, |deta| <= 1 < pi: P(related | eta_1, eta_2) = |deta|/pi, so the ordering
    fraction is E|eta_1 - eta_2|/pi with tan(eta) uniform on [-tan eta0, tan eta0] (rho = sec^2 eta/...)."""
    from scipy import integrate
    eta0 = 0.5
    T = math.tan(eta0)
    val, _ = integrate.dblquad(lambda a, b: abs(math.atan(a) - math.atan(b)) / (4 * T * T), -T, T, -T, T)
    want = val / math.pi
    N, fr = 300, []
    for seed in range(40):
        B = oracle.link(DS, csg_inputs.sprinkle_de_sitter(N, 2000 + seed, eta0))
        fr.append(np.triu(B, 1).sum() / (N * (N - 1) / 2))
    fr = np.array(fr)
    assert abs(fr.mean() - want) <= 4 * fr.std(ddof=1) / math.sqrt(len(fr))


def test_4d_boost_invariance():
    """A Lorentz boost changes every coordinate and the time order but not who is related to whom
    (up to rounding exactly on the cone)."""
    N = 400
    c = csg_inputs.sprinkle(4, N, 77)
    B = oracle.link(M4, c)
    ch, sh = math.cosh(0.4), math.sinh(0.4)
    boosted = c.copy()
    boosted[:, 0] = ch * c[:, 0] + sh * c[:, 1]
    boosted[:, 1] = sh * c[:, 0] + ch * c[:, 1]
    order = np.argsort(boosted[:, 0], kind="stable")
    Bb = oracle.link(M4, boosted[order])
    back = np.empty_like(Bb)
    back[np.ix_(order, order)] = Bb
    assert (back != B).sum() <= 4


@pytest.mark.parametrize("geom,N,seed", [(M2, 700, 1), (M4, 700, 2), (DS, 700, 3), (M4, 1, 4), (DS, 2, 5)])
def test_generator_bitset_is_the_same_relation(geom, N, seed):
    """The seeded input generator (csg_inputs/gen.c) and the link oracle agree bit for bit, so the action tests
    and the linking tests speak about the same causal sets."""
    if geom == DS:
        coords, bits = csg_inputs.make_de_sitter(N, seed)
    else:
        coords, bits = csg_inputs.make_causet(4 if geom == M4 else 2, N, seed)
    B = oracle.link(geom, coords)
    assert (csg_inputs.pack_dense(np.triu(B, 1)) == bits).all()
