"""Host-side arithmetic of bench.py that the roofline object rests on (no GPU): the share of the dense K sweep's
two-stage groups that the block-sparse sweep executes, recomputed by bench.executed_group_fraction from the library's
occupancy map, against a literal tile-by-tile walk of the kernel's rules (tensor_kernel.cuh: tile_k_range, for_live_groups);
and useful_work_ratio against its definition."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
import csg_inputs  # noqa: E402


def occupancy_words(occ):
    nB = occ.shape[0]
    stride = (((nB + 31) // 32 + 4 + 3) // 4) * 4                      # occ_stride_words of occupancy_kernel.cuh
    w = np.zeros((nB, stride), dtype=np.uint32)
    for K in range(nB):
        w[:, K // 32] |= occ[:, K].astype(np.uint32) << np.uint32(K % 32)
    return w


def walk_tiles(occ):
    """Literal restatement: tile (I, J) sweeps stages I..J, widened to an even count (downwards if possible, else
    upwards); a group of two stages is live if one of its stages kb has occ[I][kb] and occ[J][kb] -- the kernel does not
    exempt the widening stage, whose products are all masked: a group may run for nothing, never the reverse; a tile
    keeps one group."""
    nB = occ.shape[0]
    live = dense = 0
    for I in range(nB):
        for J in range(I, nB):
            b, e = I, J + 1
            if (e - b) & 1:
                if b > 0:
                    b -= 1
                else:
                    e += 1
            groups = (e - b) // 2
            n = 0
            for g in range(groups):
                for kb in (b + 2 * g, b + 2 * g + 1):
                    if kb < nB and occ[I, kb] and occ[J, kb]:
                        n += 1
                        break
            live += max(n, 1)
            dense += groups
    return live / dense


@pytest.mark.parametrize("nB,p,seed", [(1, 1.0, 0), (2, 0.5, 1), (7, 0.6, 2), (16, 0.3, 3), (33, 0.8, 4), (40, 0.0, 5), (40, 1.0, 6)])
def test_executed_group_fraction_equals_the_literal_walk(nB, p, seed):
    rng = np.random.default_rng(seed)
    occ = rng.random((nB, nB)) < p
    occ = occ | occ.T                                                 # the relation matrix is symmetric, so is its occupancy
    got = bench.executed_group_fraction(occupancy_words(occ), 256 * nB)
    assert got == pytest.approx(walk_tiles(occ), abs=1e-12)


def test_executed_group_fraction_edge_maps():
    nB = 9
    occ = np.ones((nB, nB), dtype=bool)
    assert bench.executed_group_fraction(occupancy_words(occ), 256 * nB) == 1.0
    occ[:] = False
    occ[0, :] = occ[:, 0] = True                                      # only row/column block 0 populated
    assert bench.executed_group_fraction(occupancy_words(occ), 256 * nB) == pytest.approx(walk_tiles(occ), abs=1e-12)


@pytest.mark.parametrize("dim,N,seed", [(2, 300, 1), (4, 700, 2), (2, 1025, 3)])
def test_useful_work_ratio_equals_its_definition(dim, N, seed):
    _, bits = csg_inputs.make_causet(dim, N, seed)
    U = np.zeros((N, N), dtype=bool)
    for i in range(N):
        row = np.unpackbits(bits[i].view(np.uint8), bitorder="little")[:N].astype(bool)
        U[i, i + 1:] = row[i + 1:]
    ii, jj = np.nonzero(U)
    want = int((jj - ii - 1).sum()) / bench.comb3(N)
    assert bench.useful_work_ratio(bits, N) == pytest.approx(want, rel=1e-12)
