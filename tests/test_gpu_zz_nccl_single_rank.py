"""The N>1 path's collective on real hardware, as far as one GPU allows: a ONE-rank NCCL process group, in which
multigpu.csg_action_sharded runs, and the same three steps run by hand with the collective forced through NCCL
(csg_action_partial -> ncclAllReduce of the int64 abundances on the device, torch.distributed's nccl backend ->
csg_action_finish; the library call itself skips the all-reduce in a group of one).  The multi-rank logic itself (shard partition, sums) is covered
by the world_size-2 gloo tests on CPU and by the summed shards of test_gpu_parity.py; this test is there so that the
NCCL call, its dtype and its stream ordering have executed at least once on a B200.  Runs in a subprocess (its own
rendezvous on 127.0.0.1, a free port, a timeout) so that the process group never leaks into the other tests; the file
sorts late among the GPU tests because the round's end runs `pytest -x`."""
import os
import socket
import subprocess
import sys

import pytest

import csg_inputs
import oracle

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

SCRIPT = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
import csg_inputs, paper_1709_03013_b200 as csg
from paper_1709_03013_b200 import multigpu
torch.cuda.set_device(0)
try:
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    probe = torch.ones(1, dtype=torch.int64, device="cuda")
    dist.all_reduce(probe)
    torch.cuda.synchronize()
except Exception as e:                                  # no usable NCCL / rendezvous on this box: the test says so and skips
    print("NCCL_UNAVAILABLE", type(e).__name__, str(e)[:300])
    sys.exit(0)
csg.load()
out = []
for dim, N, eps, kmax in ((4, 2700, 1.0, 3), (2, 5000, 0.1, 4998)):
    _, bits = csg_inputs.make_causet(dim, N, 12 + N)
    d = csg.to_device(bits)
    c1, S1 = multigpu.csg_action_sharded(d, N, dim, eps, kmax)          # (skips the all-reduce in a group of one)
    c2, S2 = csg.csg_action(d, N, dim, eps, kmax)
    # the same three steps by hand with the collective forced through NCCL: int64, on the device, stream-ordered
    c3 = csg.csg_action_partial(d, N, kmax, 0, 1)
    dist.all_reduce(c3, op=dist.ReduceOp.SUM)
    S3 = csg.csg_action_finish(c3, N, dim, eps, kmax)
    torch.cuda.synchronize()
    assert torch.equal(c1, c2) and float(S1.item()) == float(S2.item()), (dim, N)
    assert torch.equal(c3, c2) and float(S3.item()) == float(S2.item()), (dim, N)
    out.append([int(x) for x in c1[:4].cpu()])
t = multigpu.max_over_ranks([1.5, 2.5], device="cuda")
assert [float(x) for x in t] == [1.5, 2.5]
m = torch.tensor([1.5, 2.5], dtype=torch.float64, device="cuda")
dist.all_reduce(m, op=dist.ReduceOp.MAX)                              # the timing reduction of bench.py, through NCCL
assert m.tolist() == [1.5, 2.5]
dist.barrier()
dist.destroy_process_group()
print("NCCL_SINGLE_RANK_OK", out)
"""


def test_sharded_action_through_a_one_rank_nccl_group():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", SCRIPT, root], capture_output=True, text=True, timeout=300, env=env)
    if "NCCL_UNAVAILABLE" in r.stdout:
        pytest.skip("NCCL could not be brought up in a one-rank group here: " + r.stdout[-400:])
    assert r.returncode == 0 and "NCCL_SINGLE_RANK_OK" in r.stdout, (r.returncode, r.stdout[-500:], r.stderr[-2000:])
    _, bits = csg_inputs.make_causet(4, 2700, 12 + 2700)
    want = oracle.alg5_counts(bits, 2700, 3)
    assert str([int(x) for x in want]) in r.stdout
