"""Writes tests/golden/config_histograms.txt: for the BASELINE.json configs whose reference histogram takes
minutes (configs 2, 3, 4), the interval-abundance histogram computed by the ORACLE ONLY (Algorithm 5 restated,
oracle/alg5_packed.c, pinned bit for bit to the plain triple loop in tests/test_oracle_pins.py), stored as
    name N kmax bitset_fnv1a64 sha256(counts as little-endian int64) sum(counts) counts[0..7]
so that GPU parity tests can check the FULL histogram of a config without re-running minutes of CPU work.
Nothing here touches the CUDA path.  Usage: python tests/golden/make_config_goldens.py [config indices]"""
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


def line_for(index):
    cfg = csg_inputs.CONFIGS[index]
    N = cfg["N"]
    _, bits = csg_inputs.make_config(cfg)
    t0 = time.time()
    counts = oracle.alg5_counts(bits, N, N - 2)          # full histogram, k = 0..N-2
    sha = hashlib.sha256(np.ascontiguousarray(counts, dtype="<i8").tobytes()).hexdigest()
    head = " ".join(str(int(c)) for c in counts[:8])
    print("config %d done in %.0f s" % (index, time.time() - t0), file=sys.stderr)
    return "%s %d %d %016x %s %d %s" % (cfg["name"], N, N - 2, csg_inputs.bits_hash(bits), sha, int(counts.sum()), head)


if __name__ == "__main__":
    todo = [int(a) for a in sys.argv[1:]] or [2, 3, 4]
    old = {}
    if os.path.exists(OUT):
        for ln in open(OUT):
            if ln.strip() and not ln.startswith("#"):
                old[ln.split()[0]] = ln.strip()
    for i in todo:
        ln = line_for(i)
        old[ln.split()[0]] = ln
    with open(OUT, "w") as f:
        f.write("# written by tests/golden/make_config_goldens.py (oracle only): name N kmax bitset_fnv1a64 sha256 sum counts[0..7]\n")
        for name in sorted(old):
            f.write(old[name] + "\n")
