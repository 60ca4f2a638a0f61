"""The seeded input generator: layout contract and recipe (reading A17)."""
import numpy as np
import pytest

import csg_inputs


def unpack(bits, N):
    by = np.ascontiguousarray(bits).view(np.uint8)
    return np.unpackbits(by, axis=1, bitorder="little")[:, : bits.shape[1] * 64]


@pytest.mark.parametrize("dim,N", [(2, 1), (2, 2), (2, 257), (4, 300), (4, 1000)])
def test_layout_contract(dim, N):
    coords, bits = csg_inputs.make_causet(dim, N, 42)
    assert bits.shape == (N, csg_inputs.stride_words(N)) and bits.dtype == np.uint64
    assert bits.shape[1] % 4 == 0                      # 256-bit aligned rows
    full = unpack(bits, N)
    assert full[:, N:].sum() == 0                      # zero padding
    B = full[:, :N]
    assert (B == B.T).all() and B.diagonal().sum() == 0
    if dim == 2:
        u, v = coords[:, 0], coords[:, 1]
        ref = (u[:, None] < u[None, :]) & (v[:, None] < v[None, :])
        assert (np.diff(u + v) >= 0).all()
    else:
        d = coords[None, :, :] - coords[:, None, :]
        s2 = d[..., 1] * d[..., 1] + d[..., 2] * d[..., 2]
        s2 = s2 + d[..., 3] * d[..., 3]
        ref = (d[..., 0] > 0) & (d[..., 0] * d[..., 0] > s2)
        assert (np.diff(coords[:, 0]) >= 0).all()
        t, r2 = coords[:, 0], (coords[:, 1:] ** 2).sum(1)
        assert (r2 < np.minimum(t, 1 - t) ** 2).all()  # inside the Alexandrov interval
    assert (np.tril(ref) == 0).all()                   # i precedes j only if i < j (time sorted)
    assert (np.triu(B, 1) == ref).all()


def test_seeded_and_distinct():
    _, a = csg_inputs.make_causet(2, 500, 1)
    _, b = csg_inputs.make_causet(2, 500, 1)
    _, c = csg_inputs.make_causet(2, 500, 2)
    assert csg_inputs.bits_hash(a) == csg_inputs.bits_hash(b) != csg_inputs.bits_hash(c)


def test_ordering_fractions():
    """2D diamond: 1/2; 4D diamond: about 0.10 (DESIGN.md input recipe)."""
    _, b2 = csg_inputs.make_causet(2, 2000, 3)
    _, b4 = csg_inputs.make_causet(4, 2000, 3)
    f2 = unpack(b2, 2000).sum() / (2000 * 1999)
    f4 = unpack(b4, 2000).sum() / (2000 * 1999)
    assert abs(f2 - 0.5) < 0.03 and abs(f4 - 0.10) < 0.02


def test_pack_dense_roundtrip():
    up, bits = csg_inputs.random_poset_bits(130, 0.2, seed=0)
    B = unpack(bits, 130)[:, :130]
    assert (np.triu(B, 1) == up).all() and (B == B.T).all()


def test_golden_histogram_file_is_what_the_oracle_writes():
    """tests/golden/config_histograms.txt (used by the GPU parity tests at the large configs) is the output of
    tests/golden/make_config_goldens.py, which calls only the oracle: regenerate the cheap line (config 1) and
    compare; check that every line is tied to the bitset the generator produces for that config name."""
    import importlib.util
    import os
    here = os.path.dirname(os.path.abspath(__file__))
    spec = importlib.util.spec_from_file_location("make_config_goldens", os.path.join(here, "golden", "make_config_goldens.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    stored = {ln.split()[0]: ln.strip() for ln in open(mod.OUT) if ln.strip() and not ln.startswith("#")}
    assert mod.line_for(1) == stored[csg_inputs.CONFIGS[1]["name"]]
    names = {c["name"]: c for c in csg_inputs.CONFIGS}
    for name, ln in stored.items():
        f = ln.split()
        assert name in names and int(f[1]) == names[name]["N"] and int(f[2]) == names[name]["N"] - 2
        assert len(f[4]) == 64 and int(f[5]) >= sum(int(x) for x in f[6:14])
