"""N > 1 host logic of bench.py on CPU: world size 2 over gloo (no GPU).

The path shards by slot ownership with no data-path collective (S8): every rank
owns its own slots and descriptor sets, the job's time is the max over ranks, the job's
value is all ranks' bytes over that time.  Each rank here runs its shard through the CPU
oracle (tests may) so that the per-rank counters and the aggregation are checked together.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        from oracle import Oracle
        w = bench.make_workload("bulk_small", rank)
        o = Oracle()
        ids = [o.slot_register(w.slot_image(s)) for s in range(len(w.slot_sizes))]
        for e in w.epochs:
            assert o.memcpy_batch(e)[0] == 0 and o.fence() == 0
        sent = sum(o.slot_counters(s)[0] for s in ids)
        fake_ms = 10.0 * (rank + 1)                       # rank 1 is the slow one
        ms_max = bench.rank_max(fake_ms, dist, "cpu")
        digest = int(np.bitwise_xor.reduce(w.epochs[0]["dst_off"].astype(np.uint64)))
        gathered = [None] * world
        dist.all_gather_object(gathered, (sent, digest, bench.bytes_per_step(w), bench.descs_per_step(w)))
        if rank == 0:
            torch.save({"ms_max": ms_max, "gathered": gathered}, out)
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_ranks_shard_and_aggregate(tmp_path):
    out = str(tmp_path / "r0.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    r = torch.load(out, weights_only=False)
    assert r["ms_max"] == 20.0                                       # max over ranks, not rank 0's own
    (s0, d0, b0, n0), (s1, d1, b1, n1) = r["gathered"]
    assert s0 == s1 == 4 * 1024                                      # every rank fenced its own 4 sets
    assert d0 != d1                                                  # different seeds: different tables
    import bench
    agg = bench.shard_report([b0 * 4, b1 * 4], [n0 * 4, n1 * 4], r["ms_max"], 4)
    assert agg["value"] == pytest.approx((b0 + b1) * 4 / 20e-3 / 1e9)
    assert agg["descs_per_s"] == pytest.approx((n0 + n1) * 4 / 20e-3)
    assert agg["ms_per_step"] == 5.0


def test_rank_max_single_process():
    import bench
    assert bench.rank_max(3.5) == 3.5


def test_gpus_flag_without_a_launcher_starts_the_ranks(monkeypatch):
    """`python bench.py --gpus N` on its own must not run one rank and call it N: without
    WORLD_SIZE in the environment it re-launches itself as N ranks with the contract's line."""
    import subprocess

    import bench
    cmd = bench.spawn_command(4, ["--gpus", "4", "--steps", "5"], port=29511)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"]
    assert cmd[cmd.index("--nproc-per-node") + 1] == "4"
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29511"
    assert cmd[-5:] == [os.path.join(ROOT, "bench.py"), "--gpus", "4", "--steps", "5"]
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    seen = []
    monkeypatch.setattr(subprocess, "call", lambda c: seen.append(c) or 0)
    monkeypatch.setattr(torch.cuda, "device_count", lambda: 2)
    assert bench.main(["--gpus", "2", "--steps", "3", "--warmup", "3"]) == 0
    assert len(seen) == 1 and seen[0][-6:] == ["--gpus", "2", "--steps", "3", "--warmup", "3"]
    with pytest.raises(SystemExit) as e:
        bench.main(["--gpus", "8"])                      # more ranks than devices: refused, not shrunk
    assert "8" in str(e.value) and not seen[1:]
