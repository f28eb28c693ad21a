"""The spike exchange of the target-sharded mode ACROSS PROCESSES: two processes, one handle each, both on cuda:0, the
receive buffers mapped into the peer process through CUDA IPC handles (ng_exchange_handle / ng_exchange_attach,
binding.connect_peers over gloo).  One GPU cannot run two ranks' kernels at the same time, so no kernel may wait for
another (B200_PROFILING.md): the ranks issue every step in two halves with a host barrier in between — update + publish,
barrier, gather + deliver — so that each flag is set before its gather starts.  The peer stores, flags, counts and the
gather are the code a multi-GPU run uses; only the waiting is done on the host here.
Rank 0 compares the whole network's spike record with a one-GPU run of the same seeded network."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
from paper_2007_14236_b200 import binding as B, workloads as W
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
wl = W.microcircuit(scale_div=40, n_steps=120, indegree_div=8)
v0 = wl.initial_v()
g = B.Sim(0.1, wl.ring_slots, wl.seed, record_spikes=True, rank=rank, world=world)
wl.apply(g); g.prepare()
B.connect_peers(g, dist)
f0, n = B.shard_range(wl.n_neurons, rank, world)
g.set_state(B.FIELD_V, v0[f0:f0 + n])
steps = 120
for _ in range(steps):
    g.shard_phase(0); g.stream.synchronize(); dist.barrier()
    g.shard_phase(1); g.stream.synchronize(); dist.barrier()
s, i = g.get_spikes()
assert g.get_state(B.FIELD_STEP) == steps
if rank == 0:
    one = B.Sim(0.1, wl.ring_slots, wl.seed, record_spikes=True)
    wl.apply(one); one.prepare(); one.set_state(B.FIELD_V, v0)
    one.set_option(B.OPT_DELIVERY_KERNEL, 1); one.set_option(B.OPT_STEP_MODE, 0)
    one.simulate(steps)
    s1, i1 = one.get_spikes()
    a = set(zip(s.tolist(), i.tolist())); b = set(zip(s1.tolist(), i1.tolist()))
    first = 60
    a0 = {x for x in a if x[0] < first}; b0 = {x for x in b if x[0] < first}
    assert len(b0) > 100 and len(a0 ^ b0) <= 2, (len(a0), len(b0), sorted(a0 ^ b0)[:5])
    assert abs(len(a) - len(b)) <= 0.1 * len(b) + 5, (len(a), len(b))
    one.close()
# every rank recorded the whole network's spikes: compare the counts across ranks
cnt = [None] * world
dist.all_gather_object(cnt, int(s.size))
assert len(set(cnt)) == 1, cnt
dist.barrier()
g.close()
dist.destroy_process_group()
sys.stdout.write("ok %d\n" % rank); sys.stdout.flush()
'''


def test_two_processes_exchange_spikes_through_cuda_ipc(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29641", str(script), ROOT]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, (out.stdout[-1500:], out.stderr[-3000:])
    assert "ok 0" in out.stdout and "ok 1" in out.stdout
