"""Pins of the oracle against things other than itself (all CPU, -m "not gpu").

Each test names the pin (P-numbers of SURVEY.md 8c / DESIGN.md "Oracle pins") and what mistake it catches.
"""
import itertools
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import csg_inputs
import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def upper_from_bits(bits, N):
    B = oracle.expand(bits, N)
    return np.triu(B, 1).astype(np.int64)


def hist_from_matrix_square(up, kmax):
    """Library-routine route: for a symmetric relation matrix with strict upper part U, (U @ U)[i, j] =
    sum_k U[i,k] U[k,j] counts exactly the k with i<k<j related to both (U is strictly triangular, so the
    range restriction is implicit) -- an integer matmul instead of the oracle's triple loop."""
    U = up.astype(np.int64)
    C = U @ U
    vals = C[U == 1]
    h = np.bincount(vals, minlength=kmax + 1)[: kmax + 1] if vals.size else np.zeros(kmax + 1, np.int64)
    return h.astype(np.int64)


def brute_force_triples(up):
    """Tiny-input brute force: enumerate every ordered triple i<k<j with three relation look-ups."""
    N = up.shape[0]
    rel = {(i, j) for i in range(N) for j in range(i + 1, N) if up[i, j]}
    counts = {}
    for (i, j) in rel:
        n = sum(1 for k in range(i + 1, j) if (i, k) in rel and (k, j) in rel)
        counts[n] = counts.get(n, 0) + 1
    return counts


# ---------------------------------------------------------------- P1: brute force + matmul identity
@pytest.mark.parametrize("N", [1, 2, 3, 5, 17, 24])
@pytest.mark.parametrize("transitive", [True, False])
def test_p1_brute_force_triples(N, transitive):
    up, bits = csg_inputs.random_poset_bits(N, 0.3, seed=100 + N, transitive=transitive)
    kmax = max(N - 2, 0)
    got = oracle.counts_from_bits(bits, N, kmax)
    want = brute_force_triples(up)
    for n in range(kmax + 1):
        assert got[n] == want.get(n, 0), (N, n)
    assert sum(want.values()) == got.sum()


@pytest.mark.parametrize("N,p", [(33, 0.5), (64, 0.2), (65, 0.08), (130, 0.05), (257, 0.02)])
@pytest.mark.parametrize("transitive", [True, False])
def test_p1_matrix_square(N, p, transitive):
    up, bits = csg_inputs.random_poset_bits(N, p, seed=7 * N, transitive=transitive)
    got = oracle.counts_from_bits(bits, N, N - 2)
    want = hist_from_matrix_square(up, N - 2)
    assert (got == want).all()


def test_kmax_truncates_not_clamps():
    """Pairs with n > kmax are dropped, not folded into the last bin."""
    up, bits = csg_inputs.random_poset_bits(80, 0.2, seed=5)
    full = oracle.counts_from_bits(bits, 80, 78)
    cut = oracle.counts_from_bits(bits, 80, 3)
    assert (cut == full[:4]).all() and full[4:].sum() > 0


# ---------------------------------------------------------------- P2/P3/P4: invariants
@pytest.mark.parametrize("N,p", [(100, 0.1), (200, 0.03)])
def test_p2_p3_p4_invariants(N, p):
    up, bits = csg_inputs.random_poset_bits(N, p, seed=N)
    c = oracle.counts_from_bits(bits, N, N - 2)
    k = np.arange(N - 1)
    assert c.sum() == up.sum()                                   # I1: sum_k N_k = #relations
    indeg, outdeg = up.sum(0), up.sum(1)
    assert (k * c).sum() == int((indeg * outdeg).sum())          # I2 via I3 (transitive): 3-chains by middle


# ---------------------------------------------------------------- P7: hand posets, closed forms
def test_p7_antichain():
    N = 50
    bits = csg_inputs.pack_dense(np.zeros((N, N)))
    c = oracle.counts_from_bits(bits, N, N - 2)
    assert c.sum() == 0
    assert oracle.action_local(2, N, c) == 2.0 * N
    assert oracle.action_local(4, N, c) == (4.0 / math.sqrt(6.0)) * N


@pytest.mark.parametrize("N", [3, 4, 10, 67])
def test_p7_chain(N):
    """Total order: pair (i,j) has j-i-1 elements between => N_k = N-1-k."""
    bits = csg_inputs.pack_dense(np.triu(np.ones((N, N)), 1))
    c = oracle.counts_from_bits(bits, N, N - 2)
    assert (c == N - 1 - np.arange(N - 1)).all()
    # Eq. 4 by hand: N - 2(N-1) + 4(N-2) - 2(N-3) = N  => S = 2N   (N >= 3... N-3 >= 0)
    assert oracle.action_local(2, N, c) == 2.0 * N
    if N >= 4:
        # N - (N-1) + 9(N-2) - 16(N-3) + 8(N-4) = N - 1
        assert oracle.action_local(4, N, c) == (4.0 / math.sqrt(6.0)) * (N - 1)


def test_p7_layers():
    a, b, c3 = 4, 7, 5
    # complete 2-layer: every bottom element below every top element
    N = a + b
    up = np.zeros((N, N))
    up[:a, a:] = 1
    c = oracle.counts_from_bits(csg_inputs.pack_dense(up), N, N - 2)
    assert c[0] == a * b and c[1:].sum() == 0
    assert oracle.action_local(2, N, c) == 2.0 * (N - 2 * a * b)
    # complete 3-layer (transitively closed): N_0 = ab+bc, N_b = ac
    N = a + b + c3
    up = np.zeros((N, N))
    up[:a, a:] = 1
    up[a:a + b, a + b:] = 1
    c = oracle.counts_from_bits(csg_inputs.pack_dense(up), N, N - 2)
    want = np.zeros(N - 1, np.int64)
    want[0] = a * b + b * c3
    want[b] = a * c3
    assert (c == want).all()
    I4 = N - want[0] + 9 * want[1] - 16 * want[2] + 8 * want[3]
    assert oracle.action_local(4, N, c) == (4.0 / math.sqrt(6.0)) * I4


def test_dirty_diagonal_and_range_are_open():
    """A3: bits i and j themselves must not be counted even if the diagonal is (wrongly) set."""
    N = 70
    up, bits = csg_inputs.random_poset_bits(N, 0.2, seed=9)
    ref = oracle.counts_from_bits(bits, N, N - 2)
    dirty = bits.copy()
    for r in range(N):
        dirty[r, r // 64] |= np.uint64(1) << np.uint64(r % 64)
    assert (oracle.counts_from_bits(dirty, N, N - 2) == ref).all()


# ---------------------------------------------------------------- P8/P9: all N! 2D orders, exact rationals
def expected_counts_closed_form(N):
    """P9.  Two points of a random 2D order are related w.p. 1/2; given that, their rectangle has sides
    a,b with density 2(1-a)*2(1-b); each of the other N-2 points falls inside w.p. ab.  Expanding
    (1-ab)^m and integrating gives the formula in tests/golden/p8_expected_counts_2d_orders.txt."""
    out = []
    for k in range(N - 1):
        m = N - 2 - k
        s = sum(Fraction((-1) ** r * math.comb(m, r), ((k + r + 1) * (k + r + 2)) ** 2) for r in range(m + 1))
        out.append(Fraction(math.comb(N, 2), 2) * math.comb(N - 2, k) * 4 * s)
    return out


def load_p8_golden():
    table = {}
    with open(os.path.join(GOLDEN, "p8_expected_counts_2d_orders.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            n, vals = line.split(":")
            table[int(n)] = [Fraction(v) for v in vals.split()]
    return table


@pytest.mark.parametrize("N", [2, 3, 4, 5, 6])
def test_p8_exhaustive_2d_orders(N):
    total = np.zeros(N - 1, dtype=np.int64)
    s_total = Fraction(0)
    nperm = 0
    for perm in itertools.permutations(range(N)):
        p = np.array(perm)
        up = np.triu(p[:, None] < p[None, :], 1)      # u-order = index, v-order = perm
        c = oracle.counts_from_bits(csg_inputs.pack_dense(up), N, N - 2)
        total += c
        cc = np.concatenate([c, np.zeros(3, np.int64)])
        s = oracle.action_local(2, N, cc)
        assert s == 2 * (N - 2 * cc[0] + 4 * cc[1] - 2 * cc[2])
        s_total += Fraction(int(s))
        nperm += 1
    mean = [Fraction(int(t), nperm) for t in total]
    assert mean == load_p8_golden()[N]
    assert mean == expected_counts_closed_form(N)
    assert s_total / nperm == 2                        # E[S_2D] = 2 exactly


def test_p9_harmonic_form():
    for N in (2, 7, 30):
        H = sum(Fraction(1, i) for i in range(1, N + 1))
        assert expected_counts_closed_form(N)[0] == (N + 1) * H - 2 * N


# ---------------------------------------------------------------- P6: dominance counting from coordinates
def hist_from_coordinates_2d(coords):
    """n_ij = number of sprinkled points strictly inside the rectangle (u_i,u_j) x (v_i,v_j), from a 2D
    prefix sum over the rank grid -- no relation matrix, no AND, no popcount."""
    N = coords.shape[0]
    ru = np.argsort(np.argsort(coords[:, 0], kind="stable"), kind="stable")
    rv = np.argsort(np.argsort(coords[:, 1], kind="stable"), kind="stable")
    G = np.zeros((N + 1, N + 1), dtype=np.int32)
    G[ru + 1, rv + 1] = 1
    P = G.cumsum(0).cumsum(1)                          # P[a, b] = #points with ru < a and rv < b
    i, j = np.triu_indices(N, 1)
    lo_u, hi_u = np.minimum(ru[i], ru[j]), np.maximum(ru[i], ru[j])
    related = (ru[i] < ru[j]) == (rv[i] < rv[j])
    lo_v, hi_v = np.minimum(rv[i], rv[j]), np.maximum(rv[i], rv[j])
    n = P[hi_u, hi_v] - P[lo_u + 1, hi_v] - P[hi_u, lo_v + 1] + P[lo_u + 1, lo_v + 1]
    return np.bincount(n[related], minlength=N - 1)[: N - 1].astype(np.int64), int(related.sum())


@pytest.mark.parametrize("N,seed", [(300, 11), (1024, csg_inputs.CONFIGS[0]["seed"])])
def test_p6_dominance_counting_2d(N, seed):
    coords, bits = csg_inputs.make_causet(2, N, seed)
    want, nrel = hist_from_coordinates_2d(coords)
    got = oracle.counts_from_bits(bits, N, N - 2)
    assert got.sum() == nrel
    assert (got == want).all()


# ---------------------------------------------------------------- P5/P6 as a second oracle form: oracle/dominance2d.c
def brute_force_rectangles(coords):
    """O(N^3) from the coordinates alone: for every pair with u_a<u_b and v_a<v_b count the points strictly inside
    the rectangle.  Catches a wrong strictness, a swapped axis or an off-by-one in the prefix sums."""
    u, v = coords[:, 0], coords[:, 1]
    N = len(u)
    h = np.zeros(max(N - 1, 1), dtype=np.int64)
    for a in range(N):
        for b in range(N):
            if u[a] < u[b] and v[a] < v[b]:
                h[int(((u > u[a]) & (u < u[b]) & (v > v[a]) & (v < v[b])).sum())] += 1
    return h


@pytest.mark.parametrize("N,seed", [(2, 1), (3, 2), (7, 3), (64, 4), (211, 5)])
def test_dominance2d_against_brute_force_rectangles(N, seed):
    coords = csg_inputs.sprinkle(2, N, seed)
    rng = np.random.default_rng(seed)
    shuffled = coords[rng.permutation(N)]               # the element order must not matter
    want = brute_force_rectangles(coords)
    assert (oracle.dominance2d_counts(coords, N - 2) == want[: N - 1]).all()
    assert (oracle.dominance2d_counts(shuffled, N - 2) == want[: N - 1]).all()
    assert oracle.dominance2d_relations(shuffled) == want.sum()


@pytest.mark.parametrize("N,seed", [(1, 9), (2, 9), (257, 9), (1000, 10), (3000, 12), (1024, csg_inputs.CONFIGS[0]["seed"])])
def test_dominance2d_equals_triple_loop(N, seed):
    """The coordinate route and the definition on the relation matrix give the same histogram."""
    coords, bits = csg_inputs.make_causet(2, N, seed)
    kmax = max(N - 2, 0)
    want = oracle.counts_from_bits(bits, N, kmax)
    assert (oracle.dominance2d_counts(coords, kmax) == want).all()
    assert oracle.dominance2d_relations(coords) == want.sum()
    if N >= 257:                                         # kmax truncation drops exactly the higher bins
        assert (oracle.dominance2d_counts(coords, 5) == want[:6]).all()


def test_dominance2d_equals_alg5_at_config1():
    cfg = csg_inputs.CONFIGS[1]
    coords, bits = csg_inputs.make_config(cfg)
    N = cfg["N"]
    want = oracle.alg5_counts(bits, N, N - 2)
    got = oracle.dominance2d_counts(coords, N - 2)
    assert (got == want).all()
    assert oracle.dominance2d_relations(coords) == want.sum()


def test_dominance2d_row_blocks_equal_alg5_row_blocks():
    """Split by first element: each block equals Algorithm 5 on the same rows, and the blocks add up."""
    N = 2500
    coords, bits = csg_inputs.make_causet(2, N, 77)
    total = np.zeros(N - 1, dtype=np.int64)
    for r0, r1 in [(0, 1), (1, 640), (640, 1999), (1999, N)]:
        part = oracle.dominance2d_counts_rows(coords, N - 2, r0, r1)
        want, _ = oracle.alg5_counts_rows(bits, N, N - 2, r0, r1)
        assert (part == want).all(), (r0, r1)
        total += part
    assert (total == oracle.dominance2d_counts(coords, N - 2)).all()


def test_dominance2d_hand_cases():
    # a chain along the diagonal: N_k = N-1-k; an antichain along the anti-diagonal: nothing related
    N = 9
    t = np.arange(N, dtype=np.float64) / N
    assert oracle.dominance2d_counts(np.stack([t, t], 1), N - 2).tolist() == [N - 1 - k for k in range(N - 1)]
    assert oracle.dominance2d_counts(np.stack([t, t[::-1]], 1), N - 2).sum() == 0
    assert oracle.dominance2d_relations(np.stack([t, t[::-1]], 1)) == 0
    # four corners of a square and its centre: (0,0)<(1,1) holds the centre only -> one pair with n=1; the centre
    # is linked to both; (0,1) and (1,0) are related to nothing but... (0,1) vs (1,0): unrelated
    pts = np.array([[0.0, 0.0], [1.0, 1.0], [0.5, 0.5], [0.25, 0.9], [0.9, 0.25]])
    # related pairs: 0<2, 2<1, 0<1 (n=3: holds 2, 3, 4), 0<3 (n=0), 3<1 (n=0), 0<4 (n=0), 4<1 (n=0)
    assert oracle.dominance2d_counts(pts, 3).tolist() == [6, 0, 0, 1]
    with pytest.raises(ValueError):
        oracle.dominance2d_counts(np.array([[0.1, 0.2], [0.1, 0.3]]), 0)


# ---------------------------------------------------------------- P10: statistics over seeds
def test_p10_statistics_2d_orders():
    N, seeds = 128, 120
    rel, n0, chains = [], [], []
    for s in range(seeds):
        _, bits = csg_inputs.make_causet(2, N, 5000 + s)
        c = oracle.counts_from_bits(bits, N, N - 2)
        rel.append(c.sum())
        n0.append(c[0])
        chains.append((np.arange(N - 1) * c).sum())
    rel, n0, chains = map(lambda x: np.array(x, float), (rel, n0, chains))
    sig_rel = math.sqrt(N * (N - 1) * (2 * N + 5) / 72.0)          # non-inversions of a random permutation
    assert abs(rel.mean() - math.comb(N, 2) / 2) < 4 * sig_rel / math.sqrt(seeds)
    assert abs(chains.mean() - math.comb(N, 3) / 6) < 4 * chains.std(ddof=1) / math.sqrt(seeds)
    e_n0 = float(expected_counts_closed_form(N)[0])
    assert abs(n0.mean() - e_n0) < 4 * n0.std(ddof=1) / math.sqrt(seeds)


# ---------------------------------------------------------------- P12: Eq. 4 / Eq. 5 arithmetic
def f2_paper_form_exact(i, e):
    """Eq. 5 exactly as printed, in rational arithmetic; e is the exact value of a double."""
    x = 1 - e
    return x ** i * (1 - Fraction(2 * i) * e / x + e * e * i * (i - 1) / (2 * x * x))


def test_p12_f2_eps_one_is_local_weights():
    assert [oracle.f2(k, 1.0) for k in range(6)] == [1.0, -2.0, 1.0, 0.0, 0.0, 0.0]


@pytest.mark.parametrize("eps", [0.1, 2.0 ** -6, 0.5, 0.9])
def test_p12_f2_matches_exact(eps):
    e = Fraction(eps)
    for k in [0, 1, 2, 3, 10, 57, 400, 3000]:
        exact = f2_paper_form_exact(k, e)
        scale = (1 - e) ** k * (1 + 2 * e * k / (1 - e) + e * e * k * k / (2 * (1 - e) ** 2))
        # relative 1e-12 of the term scale; 1e-290 absolute because (1-e)^k underflows in double (A14)
        assert abs(Fraction(oracle.f2(k, eps)) - exact) <= Fraction(1, 10 ** 12) * scale + Fraction(1, 10 ** 290)


def test_p12_smeared_action_exact_and_limits():
    N = 400
    _, bits = csg_inputs.make_causet(2, N, 77)
    c = oracle.counts_from_bits(bits, N, N - 2)
    # eps = 1 reduces Eq. 5 to Eq. 4
    s1, _ = oracle.action_smeared_2d(N, c, 1.0)
    assert s1 == oracle.action_local(2, N, c)
    for eps in (0.1, 2.0 ** -6):
        e = Fraction(eps)
        exact = 2 * e * (N - 2 * e * sum(int(c[k]) * f2_paper_form_exact(k, e) for k in range(N - 1)))
        s, scale = oracle.action_smeared_2d(N, c, eps)
        assert abs(Fraction(s) - exact) <= Fraction(scale) * Fraction(1, 10 ** 12)
    # Eq. 5 by hand on the 2-layer poset: only N_0 = ab is non-zero and f2(0)=1 => S = 2e(N - 2e ab)
    cc = np.zeros(9, np.int64)
    cc[0] = 12
    s, _ = oracle.action_smeared_2d(10, cc, 0.25)
    assert s == 2 * 0.25 * (10 - 2 * 0.25 * 12)


# ---------------------------------------------------------------- reading A9: smeared d=4 action (not in the paper)
def f4_bracket_form_exact(i, e):
    """f_4 in the bracketed form DESIGN.md states for reading A9, in rational arithmetic."""
    x = 1 - e
    return x ** i * (1 - Fraction(9 * i) * e / x + 8 * e * e * i * (i - 1) / (x * x)
                     - Fraction(4, 3) * e ** 3 * i * (i - 1) * (i - 2) / x ** 3)


def test_a9_f4_eps_one_is_the_local_d4_weights():
    assert [oracle.f4(k, 1.0) for k in range(7)] == [1.0, -9.0, 16.0, -8.0, 0.0, 0.0, 0.0]


@pytest.mark.parametrize("eps", [0.1, 2.0 ** -6, 0.5, 0.9])
def test_a9_f4_matches_exact(eps):
    e = Fraction(eps)
    for k in [0, 1, 2, 3, 4, 10, 57, 400, 3000]:
        exact = f4_bracket_form_exact(k, e)
        x = 1 - e
        scale = x ** k * (1 + 9 * e * k / x + 8 * e * e * k * k / (x * x) + Fraction(4, 3) * e ** 3 * k ** 3 / x ** 3)
        assert abs(Fraction(oracle.f4(k, eps)) - exact) <= Fraction(1, 10 ** 12) * scale + Fraction(1, 10 ** 290)


def test_a9_smeared_d4_action_exact_and_limits():
    N = 400
    _, bits = csg_inputs.make_causet(4, N, 78)
    c = oracle.counts_from_bits(bits, N, N - 2)
    s1, _ = oracle.action_smeared_4d(N, c, 1.0)
    assert s1 == oracle.action_local(4, N, c)              # eps = 1 is the local action (reading A8)
    for eps in (0.25, 2.0 ** -4):                           # sqrt(eps) exact in double
        e = Fraction(eps)
        bracket = N - e * sum(int(c[k]) * f4_bracket_form_exact(k, e) for k in range(N - 1))
        s, scale = oracle.action_smeared_4d(N, c, eps)
        pref = (4.0 / math.sqrt(6.0)) * math.sqrt(eps)
        assert abs(Fraction(s) - Fraction(pref) * bracket) <= Fraction(scale) * Fraction(1, 10 ** 12) + abs(Fraction(s)) * Fraction(1, 10 ** 15)


# ---------------------------------------------------------------- P13/P14: second oracle forms
@pytest.mark.parametrize("N,p,transitive", [(1, 0.5, True), (2, 0.9, True), (63, 0.3, True), (64, 0.3, False),
                                            (65, 0.2, True), (129, 0.1, False), (300, 0.05, True)])
def test_p13_alg5_equals_plain(N, p, transitive):
    _, bits = csg_inputs.random_poset_bits(N, p, seed=3 * N + 1, transitive=transitive)
    kmax = max(N - 2, 0)
    assert (oracle.alg5_counts(bits, N, kmax) == oracle.counts_from_bits(bits, N, kmax)).all()
    assert (oracle.alg5_counts(bits, N, 3) == oracle.counts_from_bits(bits, N, 3)).all()


def test_p13_alg5_equals_plain_cfg0_and_4d():
    cfg = csg_inputs.CONFIGS[0]
    _, bits = csg_inputs.make_causet(cfg["dim"], cfg["N"], cfg["seed"])
    N = cfg["N"]
    assert (oracle.alg5_counts(bits, N, N - 2) == oracle.counts_from_bits(bits, N, N - 2)).all()
    _, bits = csg_inputs.make_causet(4, 1500, 31)
    assert (oracle.alg5_counts(bits, 1500, 1498) == oracle.counts_from_bits(bits, 1500, 1498)).all()


def test_alg5_rows_partition():
    _, bits = csg_inputs.make_causet(4, 700, 8)
    full = oracle.alg5_counts(bits, 700, 698)
    a, ta = oracle.alg5_counts_rows(bits, 700, 698, 0, 250)
    b, tb = oracle.alg5_counts_rows(bits, 700, 698, 250, 700)
    assert (a + b == full).all()
    assert ta + tb == math.comb(700, 3)


def test_p14_pair_function():
    N = 200
    up, bits = csg_inputs.random_poset_bits(N, 0.1, seed=4)
    vals = []
    for i in range(N):
        for j in range(i + 1, N):
            n = oracle.pair_interval(bits, N, i, j)
            assert (n >= 0) == bool(up[i, j])
            if n >= 0:
                vals.append(n)
    assert (np.bincount(vals, minlength=N - 1) == oracle.counts_from_bits(bits, N, N - 2)).all()
    assert oracle.pair_interval(bits, N, 5, 5) == -1 and oracle.pair_interval(bits, N, 9, 3) == -1
