"""Writes tests/golden/config_histograms.txt: for the BASELINE.json configs whose reference histogram takes
minutes (configs 2, 3, 4), the interval-abundance histogram computed by the ORACLE ONLY (Algorithm 5 restated,
oracle/alg5_packed.c, pinned bit for bit to the plain triple loop in tests/test_oracle_pins.py), stored as
    name N kmax bitset_fnv1a64 sha256(counts as little-endian int64) sum(counts) counts[0..7]
so that GPU parity tests can check the FULL histogram of a config without re-running minutes of CPU work.
Nothing here touches the CUDA path.

    python tests/golden/make_config_goldens.py [config indices]      # default 2 3 4
    python tests/golden/make_config_goldens.py --alg5 4              # config 4 again by Algorithm 5 (hours)
    python tests/golden/make_config_goldens.py --check-partial 4     # finished Algorithm-5 blocks vs dominance2d

Configs 2 and 3 (4D) use Algorithm 5 (1.5 and 12 minutes on 8 cores).  Config 4 (2D, N=262144) uses the oracle's
coordinate route, oracle/dominance2d.c (every n_ij = points strictly inside the pair's rectangle, no relation
matrix; pinned to the triple loop and to Algorithm 5 in tests/test_oracle_pins.py): about 5 minutes.  The field
`via=` of a line names the route.  `--alg5` recomputes a line by Algorithm 5 on the relation matrix -- at config 4
that is hours of CPU, so the run is cut into blocks of first elements i (oracle.alg5_counts_rows; the blocks'
histograms add up to the whole one, pinned in tests/test_oracle_pins.py), every finished block is saved under
tests/golden/.partial/ (git-ignored) and an interrupted run resumes -- and REFUSES to write (exit 1) if the result
differs from a line already stored for that config; on agreement the line's field becomes via=...+alg5."""
import hashlib
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import numpy as np  # noqa: E402

import csg_inputs  # noqa: E402
import oracle  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config_histograms.txt")


def alg5_resumable(name, bits, N, block=2048):
    """Algorithm 5 over the whole set, block of rows by block of rows, each block's histogram kept on disk."""
    part = os.path.join(os.path.dirname(OUT), ".partial")
    os.makedirs(part, exist_ok=True)
    tag = "%s_%016x" % (name, csg_inputs.bits_hash(bits))
    total = np.zeros(N - 1, dtype=np.int64)
    t0 = time.time()
    for b0 in range(0, N, block):
        f = os.path.join(part, "%s_rows_%d_%d.npy" % (tag, b0, min(b0 + block, N)))
        if os.path.exists(f):
            c = np.load(f)
        else:
            c, _ = oracle.alg5_counts_rows(bits, N, N - 2, b0, min(b0 + block, N))
            np.save(f + ".tmp.npy", c)
            os.replace(f + ".tmp.npy", f)
            print("  rows %d.. done, %.0f s" % (b0, time.time() - t0), file=sys.stderr, flush=True)
        total += c
    return total


def check_partial(index):
    """Every finished Algorithm-5 block under .partial/ against the coordinate route restricted to the same first
    elements (oracle.dominance2d_counts_rows).  Prints what fraction of the related pairs that confirms."""
    cfg = csg_inputs.CONFIGS[index]
    N = cfg["N"]
    coords, bits = csg_inputs.make_config(cfg)
    part = os.path.join(os.path.dirname(OUT), ".partial")
    tag = "%s_%016x" % (cfg["name"], csg_inputs.bits_hash(bits))
    done, pairs, bad = [], 0, 0
    for fn in sorted(os.listdir(part)) if os.path.isdir(part) else []:
        if not (fn.startswith(tag + "_rows_") and fn.endswith(".npy") and ".tmp" not in fn):
            continue
        r0, r1 = (int(x) for x in fn[len(tag) + 6:-4].split("_"))
        a5 = np.load(os.path.join(part, fn))
        dom = oracle.dominance2d_counts_rows(coords, N - 2, r0, r1)
        ok = bool((a5 == dom).all())
        bad += not ok
        done.append((r0, r1))
        pairs += int(a5.sum())
        print("rows %d..%d: %s (%d related pairs)" % (r0, r1, "equal" if ok else "DIFFERENT", int(a5.sum())), flush=True)
    total = oracle.dominance2d_relations(coords)
    print("%s: %d Algorithm-5 blocks (%d rows) checked, %d differ; they hold %d of %d related pairs (%.1f %%)"
          % (cfg["name"], len(done), sum(b - a for a, b in done), bad, pairs, total, 100.0 * pairs / total))
    return bad == 0


def line_for(index, force_alg5=False):
    cfg = csg_inputs.CONFIGS[index]
    N = cfg["N"]
    coords, bits = csg_inputs.make_config(cfg)
    t0 = time.time()
    if cfg["dim"] == 2 and N > 131072 and not force_alg5:
        via = "dominance2d"
        counts = oracle.dominance2d_counts(coords, N - 2)   # full histogram, k = 0..N-2, from the coordinates
        assert int(counts.sum()) == oracle.dominance2d_relations(coords)
    elif N <= 131072:
        via = "alg5"
        counts = oracle.alg5_counts(bits, N, N - 2)
    else:
        via = "alg5"
        counts = alg5_resumable(cfg["name"], bits, N)
    sha = hashlib.sha256(np.ascontiguousarray(counts, dtype="<i8").tobytes()).hexdigest()
    head = " ".join(str(int(c)) for c in counts[:8])
    print("config %d done in %.0f s" % (index, time.time() - t0), file=sys.stderr)
    return "%s %d %d %016x %s %d %s via=%s" % (cfg["name"], N, N - 2, csg_inputs.bits_hash(bits), sha, int(counts.sum()), head, via)


if __name__ == "__main__":
    if "--check-partial" in sys.argv[1:]:
        sys.exit(0 if all([check_partial(int(a)) for a in sys.argv[1:] if not a.startswith("--")]) else 1)
    force_alg5 = "--alg5" in sys.argv[1:]
    todo = [int(a) for a in sys.argv[1:] if not a.startswith("--")] or [2, 3, 4]
    old = {}
    if os.path.exists(OUT):
        for ln in open(OUT):
            if ln.strip() and not ln.startswith("#"):
                old[ln.split()[0]] = ln.strip()
    for i in todo:
        ln = line_for(i, force_alg5)
        name = ln.split()[0]
        if force_alg5 and name in old:
            have = old[name].split()
            if have[:14] != ln.split()[:14]:
                print("MISMATCH for %s:\n  stored %s\n  alg5   %s" % (name, old[name], ln), file=sys.stderr)
                sys.exit(1)
            via = [f for f in have if f.startswith("via=")]
            if via and "alg5" not in via[0]:
                ln = " ".join(have[:14]) + " " + via[0] + "+alg5"
        old[name] = ln
    with open(OUT, "w") as f:
        f.write("# written by tests/golden/make_config_goldens.py (oracle only): name N kmax bitset_fnv1a64 sha256 sum counts[0..7] via=route\n")
        for name in sorted(old):
            f.write(old[name] + "\n")
