"""The control plane of the Global Memory Slots on CPU: two processes over gloo carry the byte
blobs of collective.exchange_global_slots / fence_global between stand-in contexts (no GPU, no
library call): every rank must hand ITS library the handles of all ranks in rank order, own
included, and the concatenated count lines of all ranks."""
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

RANK_SCRIPT = r'''
import os, sys
import numpy as np
sys.path.insert(0, %r)
import torch.distributed as dist
from paper_2509_01425_b200 import collective
from paper_2509_01425_b200.binding import GLOBAL_COUNT_DTYPE

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)

class Stub:
    """Records what the control plane hands to the local halves."""
    def global_volunteer(self, tag, key, slot):
        return bytes([rank, key, slot]) + bytes(253)
    def global_exchange(self, tag, handles):
        self.handles = list(handles)
        return [1000 + i for i in range(len(handles))]
    def global_fence_begin(self, defer_error=False):
        a = np.zeros(rank + 1, dtype=GLOBAL_COUNT_DTYPE)
        a["tag"], a["key"], a["sent"], a["recv"] = 3, np.arange(rank + 1), 10 * rank, rank
        return (a, RuntimeError("rejected batch") if rank == 1 and self.fail else None) if defer_error else a
    def global_fence_end(self, counts, timeout_ms=0):
        self.counts = np.array(counts)

s = Stub()
s.fail = False
contrib = [(10 * rank + j, 5 + j) for j in range(rank + 1)]          # rank 0 volunteers 1 slot, rank 1 two
out = collective.exchange_global_slots(s, 3, contrib)
expect = [(r, 10 * r + j, 5 + j) for r in range(world) for j in range(r + 1)]
assert [tuple(h[:3]) for h in s.handles] == expect, s.handles
assert out == {k: 1000 + i for i, (_, k, _) in enumerate(expect)}, out
collective.fence_global(s)
assert len(s.counts) == sum(r + 1 for r in range(world))
assert sorted(s.counts["sent"].tolist()) == sorted(10 * r for r in range(world) for _ in range(r + 1))
# a rank whose epoch holds a rejected batch still completes the exchange with its peers, then raises
s.fail, s.counts = True, None
try:
    collective.fence_global(s)
    raised = False
except RuntimeError:
    raised = True
assert raised == (rank == 1) and len(s.counts) == sum(r + 1 for r in range(world))
empty = collective.exchange_global_slots(s, 4, [] if rank == 0 else [(1, 2)])    # "zero or more"
assert list(empty) == [1]
dist.destroy_process_group()
print("control plane ok", rank)
''' % ROOT


def test_two_ranks_over_gloo(tmp_path):
    script = tmp_path / "rank.py"
    script.write_text(RANK_SCRIPT)
    port = 29600 + os.getpid() % 2000
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE="2", CUDA_VISIBLE_DEVICES="")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r)), stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT) for r in range(2)]
    for r, p in enumerate(procs):
        out, _ = p.communicate(timeout=300)
        assert p.returncode == 0, "rank %d:\n%s" % (r, out.decode(errors="replace")[-3000:])
        assert b"control plane ok" in out
