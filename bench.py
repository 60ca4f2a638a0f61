#!/usr/bin/env python
"""bench.py -- Benincasa-Dowker action throughput on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 0..4] [--variant 0|1|2]

One "step" = one whole pass of the hot path (csg_action: relation test, interval sizes, histogram, action) over
one synthetic causal set.  Default workload = BASELINE.json configs[3]: 4D Minkowski diamond, N = 131072
(2 GiB bitset, larger than the 126 MB L2, so no flush is needed between steps).  metric = ordered-triple tests
per second = C(N,3) / time.  N > 1 ranks (torchrun): every rank owns an independent causal set of the same
ensemble (seed + 1000*rank); no data-path collective; value = all ranks' triples / max-over-ranks time.

Prints ONE JSON line on rank 0.  `--impl reference` times the oracle (Algorithm 5 restated, oracle/alg5_packed.c)
on the host cores on a bounded sample of the same workload.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ordered_triple_tests_per_s"
UNIT = "triple-tests/s"


def comb3(n):
    return n * (n - 1) * (n - 2) // 6


def workload_name(cfg):
    what = "local action" if cfg["eps"] == 1.0 else "smeared eps=%g" % cfg["eps"]
    if cfg.get("geometry") == "ds2":
        return "(1+1) de Sitter slab eta0=%g N=%d %s (the paper's workload, PAPER.md:453-467; not a BASELINE.json config)" % (
            cfg.get("eta0", 0.5), cfg["N"], what)
    return "%dD Minkowski diamond N=%d %s (BASELINE.json configs[%d])" % (cfg["dim"], cfg["N"], what, cfg["index"])


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(bf16=float(p["bf16_tflops"]), bf16_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                    hbm=float(p["hbm_gbs"]), source="measured (MEASURED_PEAKS.json)")
    return dict(bf16=1590.0, bf16_sustained=1400.0, hbm=6650.0, source="fallback (B200_PROFILING.md)")


KERNEL_SOURCES = {"tensor_action_kernel": ["tensor_kernel.cuh"], "bitset_action_kernel": ["bitset_kernel.cuh", "finish.cuh"],
                  "link_kernel": ["link_kernel.cuh"]}


def kernel_source_hash(kernel):
    """sha256 (16 hex digits) over the source files of a kernel: profiles/dram_traffic.json records the hash its
    capture was taken at, so a capture of older code is recognised as stale."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1709_03013_b200", "csrc")
    for name in KERNEL_SOURCES[kernel.split("<")[0]]:
        h.update(open(os.path.join(csrc, name), "rb").read())
    return h.hexdigest()[:16]


def read_traffic(kernel, workload_index):
    """(dram bytes per launch, provenance) of a kernel from the committed ncu --set full summaries
    (profiles/dram_traffic.json), or (None, why): the capture must be of THIS workload and of the present sources."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.json")
    if not os.path.exists(path):
        return None, "no capture committed"
    entry = json.load(open(path)).get(kernel)
    if not isinstance(entry, dict):
        return None, "no capture committed for this kernel"
    if entry.get("config") != workload_index:
        return None, "the committed capture (%s) is of configs[%s], not of this workload" % (entry.get("capture"), entry.get("config"))
    if entry.get("csrc_sha256_16") != kernel_source_hash(kernel):
        return None, "stale: the kernel sources changed after the committed capture (%s)" % entry.get("capture")
    return entry["dram_bytes_per_launch"], "ncu --set full, %s" % entry.get("capture")


def library_gemm_context(torch):
    """Plain library GEMMs of the same box, for context beside the roofline: int8 (torch._int_mm, cuBLASLt) and
    fp8 e4m3 (torch._scaled_mm), 8192^3, best of 10 after 3 warm-ups, CUDA events.  The stack exposes no fp4 GEMM."""
    out = {}
    M = 8192

    def best_tops(fn):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        best = float("inf")
        for _ in range(10):
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        return 2.0 * M ** 3 / (best * 1e-3) / 1e12
    try:
        a = torch.randint(-3, 3, (M, M), dtype=torch.int8, device="cuda")
        b = torch.randint(-3, 3, (M, M), dtype=torch.int8, device="cuda").t()
        out["int8_torch_int_mm_tops"] = best_tops(lambda: torch._int_mm(a, b))
    except Exception as e:                                    # noqa: BLE001 -- context only
        out["int8_torch_int_mm_tops"] = "unavailable: %s" % type(e).__name__
    try:
        a8 = torch.randn(M, M, device="cuda").to(torch.float8_e4m3fn)
        b8 = torch.randn(M, M, device="cuda").to(torch.float8_e4m3fn).t()
        one = torch.tensor(1.0, device="cuda")
        out["fp8_torch_scaled_mm_tflops"] = best_tops(lambda: torch._scaled_mm(a8, b8, scale_a=one, scale_b=one, out_dtype=torch.bfloat16))
    except Exception as e:                                    # noqa: BLE001
        out["fp8_torch_scaled_mm_tflops"] = "unavailable: %s" % type(e).__name__
    out["note"] = "library GEMMs 8192^3 (burst); no fp4 GEMM in this stack -- the peak above is the kernel's own instruction, bare"
    return out


def config_dict(cfg, N, dim, eps, kmax):
    """The `config` object of the JSON line: the same keys and values from both arms (ours / reference)."""
    stride = 4 * ((N + 255) // 256)
    nbytes = N * stride * 8
    return {"workload": workload_name(cfg), "N": N, "dim": dim, "eps": eps, "kmax": kmax, "seed": cfg["seed"],
            "bitset_bytes": nbytes,
            "l2": "input (%.0f MiB) %s L2 (126 MB)" % (nbytes / 2**20, "larger than" if nbytes > 126e6 else "fits in")}


def useful_work_ratio(bits, N):
    """sum over related pairs i<j of (j-i-1), divided by C(N,3): the share of the ordered-triple tests that the paper's
    own method executes (Algorithm 5 skips unrelated pairs, PAPER.md:407 l.4-5); the dense tile formulation does all
    C(N,3).  Host side, O(N^2/64): sum_j j over the set bits of the upper triangle from word popcounts."""
    import numpy as np
    W = bits.shape[1]
    masks = [np.uint64(sum(1 << p for p in range(64) if (p >> b) & 1)) for b in range(6)]
    total = 0
    cols = np.arange(W, dtype=np.int64)
    for r0 in range(0, N, 2048):
        blk = bits[r0:min(N, r0 + 2048)].copy()
        rows = np.arange(r0, r0 + blk.shape[0], dtype=np.int64)
        wi = rows // 64
        blk[cols[None, :] < wi[:, None]] = 0                                   # words wholly left of the diagonal
        own = np.arange(blk.shape[0])
        keep = ~((np.uint64(2) << (rows % 64).astype(np.uint64)) - np.uint64(1)) if True else None
        keep = np.where(rows % 64 == 63, np.uint64(0), keep)                    # bit 63: nothing right of it in the word
        blk[own, wi] &= keep                                                    # keep columns j > i only
        pc = np.bitwise_count(blk).astype(np.int64)
        sum_j = (pc * (64 * cols)[None, :]).sum(1)
        for b in range(6):
            sum_j += (np.bitwise_count(blk & masks[b]).astype(np.int64).sum(1)) << b
        total += int((sum_j - (rows + 1) * pc.sum(1)).sum())
    return total / comb3(N) if N >= 3 else 0.0


def executed_group_fraction(occ_words, N):
    """Share of the two-stage groups of the dense K sweep that the block-sparse sweep of the fp4 kernel still executes
    (tensor_kernel.cuh: live_groups_word), from the occupancy map the library computed (csg_block_occupancy): tile (I, J)
    sweeps stages kb_begin..kb_end-1 (column blocks I..J, widened to an even count), a group of two stages is live when
    one of its stages has occupied blocks (I, kb) and (J, kb), and a tile keeps at least one group."""
    import numpy as np
    nB = (N + 255) // 256
    w = np.ascontiguousarray(occ_words).view(np.uint32)
    occ = ((w[:, :, None] >> np.arange(32, dtype=np.uint32)[None, None, :]) & 1).astype(bool).reshape(nB, -1)
    occ = np.concatenate([occ, np.zeros((nB, 2), dtype=bool)], axis=1)
    kcol = np.arange(occ.shape[1])
    dense = live = 0
    for I in range(nB):
        J = np.arange(I, nB)
        kb_begin = np.full(J.shape, I)
        kb_end = J + 1
        odd = ((kb_end - kb_begin) & 1) == 1
        kb_begin = np.where(odd & (kb_begin > 0), kb_begin - 1, kb_begin)
        kb_end = np.where(odd & (I == 0), kb_end + 1, kb_end)
        L = occ[I][None, :] & occ[J]                                              # (tiles of this row, stages)
        L &= (kcol[None, :] >= kb_begin[:, None]) & (kcol[None, :] < kb_end[:, None])
        g = np.zeros(L.shape[0], dtype=np.int64)
        for par in (0, 1):                                                        # groups start at kb_begin's parity
            rows = (kb_begin & 1) == par
            if rows.any():
                Lp = L[rows][:, par:par + 2 * ((L.shape[1] - par) // 2)]
                g[rows] = (Lp[:, 0::2] | Lp[:, 1::2]).sum(1)
        live += int(np.maximum(g, 1).sum())
        dense += int(((kb_end - kb_begin) // 2).sum())
    return live / dense if dense else 1.0


# ------------------------------------------------------------------------------------------- clocks sampler
class ClockSampler:
    """nvidia-smi sampling of SM clock and throttle reasons while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu_index = gpu_index
        self.proc = None
        self.tmp = None

    def start(self):
        try:
            self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu_index), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.tmp.flush()
        self.tmp.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.tmp.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        self.tmp.close()
        os.unlink(self.tmp.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------- oracle legs
def oracle_sample(bits, N, kmax, target_s, nblocks=16):
    """Time Algorithm 5 (oracle/alg5_packed.c, all host threads) on `nblocks` row blocks spread evenly over
    the causal set, sized from a calibration block so that the whole sample takes about target_s seconds.
    Returns (triple tests covered, seconds, rows, threads)."""
    import oracle
    oracle.build()
    t0 = time.perf_counter()
    # calibration: one row per host thread from each of 4 places
    tests = 0
    for b in range(4):
        r0 = min(N - 1, (2 * b + 1) * N // 8)
        _, t = oracle.alg5_counts_rows(bits, N, kmax, r0, min(N, r0 + oracle.alg5_threads()))
        tests += t
    dt = max(time.perf_counter() - t0, 1e-4)
    rate = tests / dt
    total_rows = 0
    want_tests = rate * target_s
    # rows per block so that the blocks together stand for ~want_tests (mean row stands for ~N^2/6 tests)
    per_row = max(1.0, N * N / 6.0)
    rows_per_block = int(max(1, min(N // nblocks, want_tests / per_row / nblocks)))
    t0 = time.perf_counter()
    tests = 0
    for b in range(nblocks):
        r0 = (2 * b + 1) * N // (2 * nblocks)
        r1 = min(N, r0 + rows_per_block)
        _, t = oracle.alg5_counts_rows(bits, N, kmax, r0, r1)
        tests += t
        total_rows += r1 - r0
    dt = time.perf_counter() - t0
    return tests, dt, total_rows, oracle.alg5_threads()


def plain_oracle_sample(bits, N, kmax, n_sub=3072):
    """The plain single-thread triple loop (oracle/csg_oracle.c) on the sub-causal-set made of the first n_sub
    elements of the workload (an order-ideal of the same sprinkling)."""
    import numpy as np
    import oracle
    n = min(N, n_sub)
    sub = np.ascontiguousarray(bits[:n])
    B = oracle.expand(sub, n)
    t0 = time.perf_counter()
    oracle.counts_plain(B, min(kmax, max(n - 2, 0)))
    dt = time.perf_counter() - t0
    return comb3(n), dt, n


def run_reference(args, cfg, rank, world):
    if rank != 0:
        return 0
    import csg_inputs
    csg_inputs.build()
    N, dim, kmax = cfg["N"], cfg["dim"], cfg["kmax"]
    _, bits = csg_inputs.make_config(cfg)
    per_step_s = 4.0
    for _ in range(args.warmup):
        oracle_sample(bits, N, kmax, 0.5, nblocks=4)
    tests_total, secs_total, rows, threads = 0, 0.0, 0, 1
    for _ in range(args.steps):
        tests, dt, r, threads = oracle_sample(bits, N, kmax, per_step_s)
        tests_total += tests; secs_total += dt; rows += r
    value = tests_total / secs_total
    sample = ("Algorithm 5 (oracle/alg5_packed.c) on %d rows per step in 16 evenly spaced row blocks of the same "
              "causal set; tests = sum over visited pairs of (j-i-1)" % (rows // max(args.steps, 1)))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs_total / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u64 bit ops (host)", "data": "synthetic",
        "config": config_dict(cfg, N, dim, cfg["eps"], kmax),
        "note": "each step is a bounded sample of the workload",
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                         "full_config_s_extrapolated": comb3(N) / value},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------- our arm
def run_ours(args, cfg, rank, local_rank, world):
    import numpy as np
    import torch
    import csg_inputs
    import paper_1709_03013_b200 as csg
    from paper_1709_03013_b200 import multigpu

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libcsg has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    # `--shard tiles` under torchrun with ONE rank still takes the sharded code path (partial -> all-reduce -> finish in a
    # one-rank NCCL group): all that a single GPU can show of it
    under_torchrun = "RANK" in os.environ and "MASTER_ADDR" in os.environ
    if world > 1 or (args.shard == "tiles" and under_torchrun):
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if csg._build.needs_build():
        if local_rank == 0:
            csg.build()
        if dist is not None:
            dist.barrier()
    csg.load()
    csg_inputs.build()
    csg.csg_set_variant(args.variant)
    csg.csg_set_host_pipeline(csg.HOST_PIPELINE_CHUNKED if args.host_pipeline == "chunked" else csg.HOST_PIPELINE_AUTO)

    N, dim, eps, kmax = cfg["N"], cfg["dim"], cfg["eps"], cfg["kmax"]
    tiles_mode = args.shard == "tiles" and dist is not None
    seed = cfg["seed"] if tiles_mode else multigpu.ensemble_seed(cfg["seed"], rank)
    t0 = time.perf_counter()
    coords, bits = csg_inputs.make_config(cfg, seed)
    gen_s = time.perf_counter() - t0
    host = torch.from_numpy(bits.view(np.int64)).pin_memory()
    d_bits = host.to("cuda", non_blocking=False)
    counts = torch.empty(kmax + 1, dtype=torch.int64, device="cuda")
    S = torch.empty(1, dtype=torch.float64, device="cuda")
    variant = csg.csg_effective_variant(N)
    kernel_name = {csg.VARIANT_BITSET: "bitset_action_kernel", csg.VARIANT_TENSOR: "tensor_action_kernel<KIND_I8>",
                   csg.VARIANT_TENSOR_FP4: "tensor_action_kernel<KIND_FP4>"}[variant]

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        if tiles_mode:      # one causal set, tiles split over the ranks, one all-reduce of the abundances
            multigpu.csg_action_sharded(d_bits, N, dim, eps, kmax, counts, S)
        else:               # one causal set per rank
            csg.csg_action(d_bits, N, dim, eps, kmax, counts, S)

    # ---- device-resident leg
    csg.csg_set_kernel_timing(True)
    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    launches0 = csg.csg_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    launches = csg.csg_launch_count() - launches0
    launches_per_step = launches // max(args.steps, 1)
    ms_total = ev0.elapsed_time(ev1)
    kernel_ms = csg.csg_kernel_ms_history(min(args.steps, 64))
    csg.csg_set_kernel_timing(False)
    result_counts = counts.cpu().numpy().copy()
    result_S = float(S.item())

    # ---- end-to-end leg: HOST buffers through csg_action_host (H2D of the bitset + D2H of counts, S inside)
    e2e_steps = max(1, min(args.steps, 5))
    csg.csg_action_host(host, N, dim, eps, kmax)   # warm-up (allocates the library's device buffers)
    barrier()
    e2e_each = []
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        t1 = time.perf_counter()
        c_host, S_host = csg.csg_action_host(host, N, dim, eps, kmax)
        e2e_each.append(1e3 * (time.perf_counter() - t1))
    e2e_s = time.perf_counter() - t0
    checks = {"e2e_equals_device": bool((c_host == result_counts).all() and S_host == result_S)}

    # ---- linking leg: coordinates -> relation matrix on the device, then coordinates -> action
    geom = (csg.GEOM_DESITTER_2D if cfg.get("geometry") == "ds2" else
            csg.GEOM_MINKOWSKI_4D if dim == 4 else csg.GEOM_MINKOWSKI_2D)
    coords_pinned = torch.from_numpy(coords).pin_memory()
    d_coords = coords_pinned.to("cuda")
    d_linked = torch.empty_like(d_bits)
    csg.csg_set_kernel_timing(True)
    link_ms = []
    for it in range(args.warmup + args.steps):
        csg.csg_link(d_coords, N, geom, d_linked)
        torch.cuda.synchronize()
        if it >= args.warmup:
            link_ms.append(csg.csg_last_link_ms())
    csg.csg_set_kernel_timing(False)
    checks["linked_matrix_equals_generator"] = bool(torch.equal(d_linked, d_bits))
    del d_linked
    csg.csg_causet_action_host(coords_pinned, N, geom, eps, kmax)   # warm-up (library-owned matrix buffer)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        c2_host, S2_host = csg.csg_causet_action_host(coords_pinned, N, geom, eps, kmax)
    e2e_coords_s = time.perf_counter() - t0
    checks["coords_in_equals_device"] = bool((c2_host == result_counts).all() and S2_host == result_S)
    if tiles_mode:
        # the all-reduced histogram of the sharded run must equal the one this GPU computes alone (same seed)
        c_single, S_single = csg.csg_action(d_bits, N, dim, eps, kmax)
        torch.cuda.synchronize()
        checks["sharded_equals_single"] = bool((c_single.cpu().numpy() == result_counts).all() and float(S_single.item()) == result_S)
    for name, ok in checks.items():
        if not ok:
            print("bench.py: CHECK FAILED: %s" % name, file=sys.stderr, flush=True)

    # ---- batched small sets: 64 causal sets of BASELINE.json configs[0]'s shape in one call
    batch_leg = None
    if rank == 0 and not args.no_batch_leg:
        c0, nb = csg_inputs.CONFIGS[0], 64
        sets = np.stack([csg_inputs.make_causet(c0["dim"], c0["N"], c0["seed"] + 7919 * (b + 1))[1] for b in range(nb)])
        d_sets = torch.from_numpy(sets.view(np.int64)).to("cuda")
        bc = torch.empty((nb, c0["kmax"] + 1), dtype=torch.int64, device="cuda")
        bS = torch.empty(nb, dtype=torch.float64, device="cuda")
        for _ in range(args.warmup):
            csg.csg_action_batch(d_sets, c0["N"], nb, c0["dim"], 1.0, c0["kmax"], bc, bS)
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        b0.record()
        for _ in range(args.steps):
            csg.csg_action_batch(d_sets, c0["N"], nb, c0["dim"], 1.0, c0["kmax"], bc, bS)
        b1.record()
        torch.cuda.synchronize()
        one0, one1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        one0.record()
        for _ in range(args.steps):
            for b in range(nb):
                csg.csg_action(d_sets[b], c0["N"], c0["dim"], 1.0, c0["kmax"], bc[b], bS[b:b + 1])
        one1.record()
        torch.cuda.synchronize()
        bms = b0.elapsed_time(b1) / args.steps
        # the same call on a batch large enough to fill the machine for many rounds: 512 sets
        nbig = 512
        big = np.stack([csg_inputs.make_causet(c0["dim"], c0["N"], c0["seed"] + 104729 * (b + 1))[1] for b in range(nbig)])
        d_big = torch.from_numpy(big.view(np.int64)).to("cuda")
        gc, gS = torch.empty((nbig, c0["kmax"] + 1), dtype=torch.int64, device="cuda"), torch.empty(nbig, dtype=torch.float64, device="cuda")
        for _ in range(args.warmup):
            csg.csg_action_batch(d_big, c0["N"], nbig, c0["dim"], 1.0, c0["kmax"], gc, gS)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        g0.record()
        for _ in range(args.steps):
            csg.csg_action_batch(d_big, c0["N"], nbig, c0["dim"], 1.0, c0["kmax"], gc, gS)
        g1.record()
        torch.cuda.synchronize()
        gms = g0.elapsed_time(g1) / args.steps
        del d_big
        batch_leg = {"workload": "%d causal sets, 2D N=%d, local action, one csg_action_batch call" % (nb, c0["N"]),
                     "ms_per_call": bms, "sets_per_s": nb / (bms * 1e-3),
                     "triple_tests_per_s": nb * comb3(c0["N"]) / (bms * 1e-3),
                     "ms_same_sets_one_csg_action_each": one0.elapsed_time(one1) / args.steps,
                     "batch_of_512": {"ms_per_call": gms, "sets_per_s": nbig / (gms * 1e-3),
                                      "triple_tests_per_s": nbig * comb3(c0["N"]) / (gms * 1e-3)},
                     "how": "ONE persistent launch of the fp4 tensor kernel over the tiles of all sets (csg.h: csg_action_batch)"}
        del d_sets

    ms_total, e2e_ms, e2e_coords_ms = multigpu.max_over_ranks([ms_total, 1e3 * e2e_s, 1e3 * e2e_coords_s], device="cuda")

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    triples = comb3(N)
    sets = 1 if tiles_mode else world           # causal sets the whole job finishes per step
    value = multigpu.whole_job_rate(sets * triples, args.steps, ms_total)
    e2e_value = multigpu.whole_job_rate(world * triples, e2e_steps, e2e_ms)   # the host-buffer call is per rank
    k_ms = sum(kernel_ms) / len(kernel_ms)
    kernel_triples = triples / world if tiles_mode else triples     # what one launch of rank 0 covers
    peaks = read_peaks()
    sm_clock_mhz = (clocks or {}).get("sm_mhz") or 1965.0
    traffic, traffic_src = read_traffic(kernel_name, cfg["index"])
    if variant in (csg.VARIANT_TENSOR, csg.VARIANT_TENSOR_FP4):
        # dense binary contraction on tcgen05: 1 triple test = 1 MAC = 2 ops.  peak = what the tensor cores of THIS device
        # sustain on the kernel's own instruction (csg_measure_peak: bare tcgen05.mma.cta_group::2 loop, same kind, shape
        # and operand sources, no producers), measured in this run for ~110 ms, i.e. a kernel timed alone.
        fp4 = variant == csg.VARIANT_TENSOR_FP4
        what = csg.PEAK_MMA_MXF4 if fp4 else csg.PEAK_MMA_I8
        csg.csg_measure_peak(what, 20000)
        p_ms, p_units = csg.csg_measure_peak(what, 400000)
        peak = 2.0 * p_units / (p_ms * 1e-3) / 1e12
        achieved = 2.0 * kernel_triples / (k_ms * 1e-3) / 1e12
        hw = 2.0 * (16384 if fp4 else 8192) * 148 * sm_clock_mhz * 1e6 / 1e12      # MAC/clk/SM x SMs x sampled clock
        ratio = 4.0 if fp4 else 2.0
        roofline = {"bound": "tensor", "kernel": kernel_name, "achieved": achieved, "peak": peak,
                    "unit": "TOP/s (%s)" % ("fp4 e2m1, kind::mxf4" if fp4 else "int8, kind::i8"),
                    "frac": achieved / peak,
                    "peak_source": "measured in this run: csg_measure_peak, bare tcgen05.mma.cta_group::2.kind::%s loop "
                                   "(M=N=256, %s), 400000 groups of 4 per SM pair, %.1f ms" % (
                                       "mxf4.block_scale" if fp4 else "i8", "K=64, A in TMEM" if fp4 else "K=32", p_ms),
                    "frac_of_hw": achieved / hw,
                    "hw_rate": "%d MAC/clk/SM x 148 SMs x %.0f MHz (sampled) = %.0f TOP/s" % (16384 if fp4 else 8192, sm_clock_mhz, hw),
                    "frac_of_scaled_bf16": achieved / (ratio * peaks["bf16"]),
                    "scaled_bf16": "%g x bf16 %s = %.0f TOP/s (power-capped cuBLAS figure; context only)" % (ratio, peaks["source"], ratio * peaks["bf16"]),
                    "kernel_ms": k_ms, "traffic": traffic, "traffic_source": traffic_src,
                    "library_gemm_context": library_gemm_context(torch)}
    else:
        # LOP3 AND + POPC + IADD per 32 triple tests: peak = measured issue rate of exactly that mix (csg_measure_peak)
        csg.csg_measure_peak(csg.PEAK_ALU_MIX, 2000)
        p_ms, p_units = csg.csg_measure_peak(csg.PEAK_ALU_MIX, 20000)
        peak = 32.0 * p_units / (p_ms * 1e-3) / 1e12
        achieved = kernel_triples / (k_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": kernel_name, "achieved": achieved, "peak": peak,
                    "unit": "T bit-tests/s", "frac": achieved / peak,
                    "peak_source": "measured in this run: csg_measure_peak, AND+POPC+ADD mix on 32-bit words, all SMs "
                                   "(%.1f lane-steps/clk/SM at %.0f MHz: the POPC pipe)" % (p_units / (p_ms * 1e-3) / 148 / (sm_clock_mhz * 1e6), sm_clock_mhz),
                    "kernel_ms": k_ms, "traffic": traffic, "traffic_source": traffic_src}
    if variant == csg.VARIANT_TENSOR_FP4:
        # block-sparse sweep (csg_set_sparse, AUTO: matrices of 96 MiB and more): what the tensor cores really executed
        sparse_on = N * csg.csg_row_stride_words(N) * 8 >= (96 << 20) and (dim != 2 or tiles_mode)   # CSG_SPARSE_AUTO
        frac_exec = 1.0
        if sparse_on:
            occ = csg.csg_block_occupancy(d_bits, N)
            torch.cuda.synchronize()
            frac_exec = executed_group_fraction(occ.cpu().numpy(), N)
        roofline["executed_fraction"] = frac_exec
        roofline["frac_executed"] = roofline["frac"] * frac_exec
        roofline["frac_of_hw_executed"] = roofline["frac_of_hw"] * frac_exec
        roofline["executed_note"] = ("block-sparse K sweep (occupancy pass inside the timed kernel span): two-stage groups whose "
                                     "U or L blocks are empty are neither fetched, expanded nor multiplied; executed_fraction "
                                     "of the dense sweep's groups remains; `achieved`/`frac` count all C(N,3) algorithmic "
                                     "tests, `frac_executed` = frac x executed_fraction is the tensor cores' own utilisation "
                                     "against the same measured peak (never above 1), `frac_of_hw_executed` the same against "
                                     "16384 MAC/clk/SM at the sampled clock")
    roofline["hbm_gbs_algorithmic"] = (N * csg.csg_row_stride_words(N) * 8) / (k_ms * 1e-3) / 1e9
    # what the paper's method would execute of these tests (it skips unrelated pairs, PAPER.md:407 l.4-5)
    roofline["useful_work_ratio"] = useful_work_ratio(bits, N)
    roofline["useful_work_note"] = ("sum over related pairs of (j-i-1) / C(N,3): Algorithm 5 executes only this share of the "
                                    "ordered-triple tests; the dense tiles execute all C(N,3), which is what `achieved` counts")

    cpu_baseline = None
    extra = {}
    if world == 1 and not args.no_cpu_baseline:
        tests, dt, rows, threads = oracle_sample(bits, N, min(kmax, 3) if eps == 1.0 else kmax, 12.0)
        cpu_baseline = {"value": tests / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
                        "sample": "Algorithm 5 restated (oracle/alg5_packed.c, OpenMP) on %d rows in 16 evenly spaced "
                                  "row blocks of the same causal set, %.1f s; tests = sum over visited pairs of (j-i-1)"
                                  % (rows, dt),
                        "full_config_s_extrapolated": comb3(N) / (tests / dt)}
        ptests, pdt, pn = plain_oracle_sample(bits, N, kmax)
        extra["cpu_baseline_plain"] = {"value": ptests / pdt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                       "sample": "plain triple loop (oracle/csg_oracle.c) on the first %d elements "
                                                 "of the same causal set, %.2f s" % (pn, pdt)}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong" if tiles_mode else "weak", "vs_baseline": None,
        "dtype": {csg.VARIANT_TENSOR: "u8 x u8 -> s32 (tcgen05 kind::i8)",
                  csg.VARIANT_TENSOR_FP4: "e2m1 x e2m1 -> f32, exact integers (tcgen05 kind::mxf4, unit scales)",
                  csg.VARIANT_BITSET: "u32 and/popc"}[variant],
        "data": "synthetic",
        "config": config_dict(cfg, N, dim, eps, kmax),
        "variant": {1: "bitset", 2: "tensor_i8", 3: "tensor_fp4"}[variant],
        "parallelism": ("1 causal set, tiles sharded over %d GPUs, one int64 all-reduce" % world) if tiles_mode
        else "1 causal set per GPU, no collectives",
        "host_generation_s": gen_s,
        "action_time_s": ms_total / args.steps * 1e-3,
        "kernel_ms_per_step": kernel_ms,
        "result": {"counts_head": [int(x) for x in result_counts[:4]], "S": result_S},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": N * csg.csg_row_stride_words(N) * 8,
                "d2h_bytes_per_step": (kmax + 1) * 8 + 8, "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps,
                "ms_median": sorted(e2e_each)[len(e2e_each) // 2], "ms_best": min(e2e_each),
                "what": "csg_action_host: pinned host matrix -> H2D in 64 row chunks (outside-in) + %s + D2H of counts and S"
                        % ("one launch per copy step" if args.host_pipeline == "chunked" else "one gated launch")},
        "gpu_launches": launches,
        "checks": checks,   # the legs of this run agree with each other (parity with the oracle is the tests' job)
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
    }
    l_ms = sum(link_ms) / len(link_ms)
    pairs = N * (N - 1) // 2
    # arithmetic instructions per pair test.  3+1 Minkowski: the single-precision filter (4 FADD + 1 FMUL + 3 FFMA; the
    # double-precision code only decides the ~1e-4 of the pairs next to the light cone) on the 128-lane FP32 pipe; the
    # two (1+1) geometries: DADD/DMUL/DSETP on the 64-lane FP64 pipe
    fp64_ops = {csg.GEOM_MINKOWSKI_4D: 8, csg.GEOM_MINKOWSKI_2D: 2, csg.GEOM_DESITTER_2D: 5}[geom]
    fp64_peak = (128 if geom == csg.GEOM_MINKOWSKI_4D else 64) * 148 * 1.965e9   # lanes/clk/SM x SMs x max clock
    line["link"] = {
        "kernel": "link_kernel<%s>" % {0: "GEOM_M2", 1: "GEOM_M4", 2: "GEOM_DS2"}[geom], "kernel_ms": l_ms,
        "pair_tests_per_s": pairs / (l_ms * 1e-3), "write_gbs": N * csg.csg_row_stride_words(N) * 8 / (l_ms * 1e-3) / 1e9,
        "roofline": {"bound": "alu", "achieved": pairs * fp64_ops / (l_ms * 1e-3) / 1e12, "peak": fp64_peak / 1e12,
                     "unit": "T fp32 instr/s" if geom == csg.GEOM_MINKOWSKI_4D else "T fp64 instr/s",
                     "frac": pairs * fp64_ops / (l_ms * 1e-3) / fp64_peak,
                     "peak_source": "derived: %d lanes/clk/SM x 148 SMs x 1.965 GHz (DESIGN.md 5.5)" % (128 if geom == csg.GEOM_MINKOWSKI_4D else 64),
                     "traffic": read_traffic("link_kernel<%s>" % {0: "GEOM_M2", 1: "GEOM_M4", 2: "GEOM_DS2"}[geom], cfg["index"])[0]},
        "e2e_from_coords": {"value": multigpu.whole_job_rate(world * triples, e2e_steps, e2e_coords_ms), "unit": UNIT,
                            "ms_per_step": e2e_coords_ms / e2e_steps, "h2d_bytes_per_step": N * dim * 8,
                            "d2h_bytes_per_step": (kmax + 1) * 8 + 8,
                            "what": "csg_causet_action_host: H2D coords + csg_link + csg_action + D2H"},
    }
    if batch_leg is not None:
        line["batch"] = batch_leg
    line.update(extra)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0 if all(checks.values()) else 3          # the line is printed either way; a failed cross-check fails the run


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="index into BASELINE.json configs (default 3, the headline); 5 = the paper's de Sitter workload")
    ap.add_argument("--variant", type=int, default=0, help="0 auto, 1 bitset, 2 tensor int8, 3 tensor fp4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-batch-leg", action="store_true")
    ap.add_argument("--host-pipeline", default="auto", choices=["auto", "chunked"],
                    help="csg_action_host: gated single launch (auto) or one launch per copy step (chunked; use it under ncu, "
                         "which serialises kernels and copies so that a kernel waiting for a copy never ends)")
    ap.add_argument("--shard", default="ensemble", choices=["ensemble", "tiles"],
                    help="N>1 GPUs: one causal set per rank (weak scaling, default) or one set with its tiles split")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    import csg_inputs
    cfg = dict(csg_inputs.CONFIGS[args.config])
    cfg["index"] = args.config
    if args.impl == "reference":
        return run_reference(args, cfg, rank, world)
    return run_ours(args, cfg, rank, local_rank, world)


if __name__ == "__main__":
    sys.exit(main())
