"""Host-side plumbing for more than one GPU (one process per GPU, torch.distributed).  No arithmetic of the
method lives here: the kernels behind csg_action_partial / csg_action_finish do all of it.

Two ways to use N GPUs:

* ensemble (weak scaling, the default of bench.py --gpus N): every rank owns its own causal set of the same
  ensemble -- the paper averages over ten graphs and runs Monte-Carlo chains.
  No data-path collective; only timings are reduced (max over ranks).
* tiles (strong scaling, bench.py --shard tiles): one causal set, its relation matrix replicated on every GPU,
  the pair tiles split over the ranks ("split the loop evenly" when the matrix fits everywhere),
  private histograms summed at the end by ONE all-reduce of kmax+1 int64 (NCCL over NVLink;
  at most 2 MiB, latency-bound), then the finishing kernel on every rank.
"""
import torch
import torch.distributed as dist

ENSEMBLE_SEED_STRIDE = 1000


def ensemble_seed(base_seed, rank):
    """Seed of rank's causal set in the ensemble leg: base + 1000*rank (DESIGN.md input recipe)."""
    return int(base_seed) + ENSEMBLE_SEED_STRIDE * int(rank)


def allreduce_counts(counts, group=None):
    """Sum the per-shard abundances over the ranks, in place (int64, exact in any order)."""
    assert counts.dtype == torch.int64
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(counts, op=dist.ReduceOp.SUM, group=group)
    return counts


def max_over_ranks(values, device=None, group=None):
    """Element-wise max over the ranks of a short list of floats (timings)."""
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return [float(x) for x in t.cpu()]


def whole_job_rate(units_per_step_all_ranks, steps, ms_total_max):
    """Whole-job throughput: units all ranks processed in `steps` steps / the slowest rank's time."""
    return units_per_step_all_ranks * steps / (ms_total_max * 1e-3)


def csg_action_sharded(rel_bits, N, dim, eps, kmax, counts=None, S=None, group=None):
    """One causal set over all ranks of `group`: csg_action_partial on this rank's tiles, one all-reduce of the
    abundances, csg_action_finish.  Every rank ends with the full counts and S.  Kernels run on torch's current
    stream, which is also the stream torch orders its NCCL work against."""
    from . import csg_action_partial, csg_action_finish
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    counts = csg_action_partial(rel_bits, N, kmax, rank, world, counts)
    allreduce_counts(counts, group)
    S = csg_action_finish(counts, N, dim, eps, kmax, S)
    return counts, S
