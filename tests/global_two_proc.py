"""One rank of test_two_processes_over_cuda_ipc (run by tests/test_gpu_global.py, never by pytest
collection): a HiCR instance = this process, one context on cuda:0, control plane = gloo."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def main():
    import torch
    import torch.distributed as dist

    import paper_2509_01425_b200 as hicr
    import workloads as W
    from global_common import NAMES, descs_for, oracle_run

    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    for big in (False, True):
        w = (W.global_copy_graph(world, per_buffer=24, src_bytes=1 << 20, dst_bytes=8 << 20, max_size=300000,
                                 seed=W.BASE_SEED + 9) if big else W.global_copy_graph(world, seed=W.BASE_SEED + 8))
        with hicr.Context(0, torch.cuda.current_stream().cuda_stream) as ctx:
            ctx.instance_set(rank, world)
            bufs = {k: torch.from_numpy(w.image(rank, k)).cuda() for k in NAMES}
            ids = {k: ctx.slot_register(bufs[k]) for k in NAMES}
            gg = hicr.collective.exchange_global_slots(ctx, w.tag, [(2 * rank, ids["gsrc"]), (2 * rank + 1, ids["gdst"])])
            assert len(gg) == 2 * world                                  # as many as were exchanged
            d = descs_for(w, rank, ids, gg)
            t = torch.from_numpy(d.view(np.uint8).copy()).cuda()
            ctx.memcpy_batch(t, n=len(d))
            hicr.collective.fence_global(ctx, timeout_ms=60000)
            oworld, mem, oids, og = oracle_run(w)
            assert ids == oids[rank] and gg == og[rank], (ids, oids[rank], gg, og[rank])
            for k in NAMES:
                assert bufs[k].cpu().numpy().tobytes() == mem[rank][k].tobytes(), "rank %d %s" % (rank, k)
                assert ctx.global_counters(ids[k]) == oworld.inst[rank].slot_global_counters(oids[rank][k]), k
            for s in list(ids.values()) + list(gg.values()):
                assert ctx.slot_counters(s) == oworld.inst[rank].slot_counters(s), s
            # Global-to-Global is rejected for slots of another process too
            try:
                ctx.memcpy_batch(W.make_descs([gg[2 * (1 - rank) + 1]], [gg[2 * rank]], [0], [0], [16]))
                raise SystemExit("global-to-global was accepted")
            except hicr.HicrError as e:
                assert e.status == hicr.HICR_ERR_ILLEGAL_DIRECTION
            dist.barrier()                                               # nobody unmaps what a peer still reads
    # the cross-GPU leg of bench.py --gpus N (N > 1), here between two processes on one GPU
    import bench
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream), hicr.Context(0, stream.cuda_stream) as ctx:
        ctx.instance_set(rank, world)
        r = bench.cross_gpu_leg(hicr, ctx, rank, world, None, stream, steps=3, pages=2048)
        assert r["window_equals_peer_source"] and r["owner_recv_total"] == r["owner_recv_expected"], r
        dist.barrier()
    dist.destroy_process_group()
    print("global two-process parity ok (rank %d)" % rank)


if __name__ == "__main__":
    main()
