"""Host-side logic of the target-sharded multi-GPU path (-m "not gpu"): the id partition (ng_shard_range, pure
arithmetic in libng.so), the restriction of the connection structure to a shard's targets (on the oracle's list), and the
multi-process plumbing of the spike exchange (binding.connect_peers) over world-size-2 gloo."""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2007_14236_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_ranges_tile_the_id_space():
    from paper_2007_14236_b200 import binding as B
    for n in (1, 7, 1000, 7718, 77169, 1_000_000, 2_000_000_000):
        for world in (1, 2, 3, 8, 16):
            nxt = 0
            sizes = []
            for r in range(world):
                first, cnt = B.shard_range(n, r, world)
                assert first == nxt and cnt >= 0
                nxt = first + cnt; sizes.append(cnt)
            assert nxt == n and max(sizes) - min(sizes) <= 1
    for bad in ((10, 2, 2), (10, -1, 2), (10, 0, 0), (10, 0, 17), (-1, 0, 1)):
        with pytest.raises(B.NgError):
            B.shard_range(*bad)


def test_restriction_to_targets_partitions_the_oracle_structure(oracle_mod):
    """What every shard must hold (checked against the GPU build in tests/test_gpu_sharded.py): the oracle's connections
    with the target in the shard's range.  The ranges partition the list, and for the fixed in-degree rule every target
    keeps its full in-degree on exactly one shard."""
    from paper_2007_14236_b200 import binding as B
    wl = W.microcircuit(scale_div=40, n_steps=10, indegree_div=8)
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed); wl.apply(o); o.prepare()
    src, tgt, w, d, ro = o.get_connections()
    N = wl.n_neurons
    indeg = np.bincount(tgt, minlength=N)
    for world in (2, 3, 5):
        seen = np.zeros(tgt.size, bool)
        for r in range(world):
            f0, n = B.shard_range(N, r, world)
            mine = (tgt >= f0) & (tgt < f0 + n)
            assert not np.any(seen & mine)
            seen |= mine
            assert np.array_equal(np.bincount(tgt[mine] - f0, minlength=n), indeg[f0:f0 + n])
        assert seen.all()


_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
from paper_2007_14236_b200 import binding as B
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
class FakeSim:                      # the two calls connect_peers makes on a handle, without a device
    def __init__(self): self.rank, self.world, self.attached = rank, world, {}
    def exchange_handle(self): return bytes([rank]) * 64, 0x1000 * (rank + 1)
    def exchange_attach(self, q, ipc_handle=None, ptr=None): self.attached[q] = ipc_handle
s = FakeSim()
B.connect_peers(s, dist)
assert set(s.attached) == set(range(world)) - {rank}, s.attached
for q, h in s.attached.items():
    assert h == bytes([q]) * 64
first, n = B.shard_range(7718, rank, world)
tot = [None] * world
dist.all_gather_object(tot, (first, n))
assert tot[0][0] == 0 and tot[-1][0] + tot[-1][1] == 7718 and all(tot[k][0] + tot[k][1] == tot[k + 1][0] for k in range(world - 1))
dist.barrier(); dist.destroy_process_group()
sys.stdout.write("ok %d\n" % rank); sys.stdout.flush()
'''


def test_exchange_plumbing_world_size_2_gloo(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29631", str(script), ROOT]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=240)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "ok 0" in out.stdout and "ok 1" in out.stdout
