"""Small end-to-end run of every kernel of the library, for compute-sanitizer (SURVEY.md S5:
"run parity tests under compute-sanitizer: memcheck, racecheck for the shared-memory staging,
synccheck for mbarriers").  Not collected by pytest; profiles/r02_sanitizer.md names the commands:

    compute-sanitizer --tool memcheck  python tests/sanitizer_target.py
    compute-sanitizer --tool racecheck python tests/sanitizer_target.py
    compute-sanitizer --tool synccheck python tests/sanitizer_target.py

Every result is compared with the oracle, so a sanitizer-clean run is also a parity run."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def main():
    import torch

    import __graft_entry__ as entry
    import oracle
    import paper_2509_01425_b200 as hicr
    import workloads as W
    from global_common import NAMES, descs_for, oracle_run
    from oracle import Oracle
    from parity import assert_same, run_gpu, run_oracle

    torch.cuda.set_device(0)
    entry.smoke()                                                    # engine (host + device tables), push / pop, pipe kernel

    # every (dst, src) alignment pair mod 16 with ragged sizes, small and large classes, TMA chunks included
    w = W.heavy_tailed("a", n_slots=4, slot_bytes=8 * W.MiB, src_zone=W.MiB, n_desc=800, smax=600 * W.KiB, seed=W.BASE_SEED + 1)
    assert_same(w, run_oracle(w), run_gpu(w, device_tables=True), "mixed sizes")
    w = W.chained_epochs(n_epochs=3, n_desc=3000, slot_bytes=4 * W.MiB)
    assert_same(w, run_oracle(w), run_gpu(w, device_tables=True), "team-sized")
    assert_same(w, run_oracle(w), run_gpu(w, device_tables=False, split=3), "host tables")

    # non-locking MPSC through the bulk-copy pipeline (aligned) and through the vector kernels (T = 24), locking MPSC
    for (P, N, T, C, mb) in ((5, 3000, 64, 64, 48), (3, 500, 24, 16, 5)):
        cw = W.mpsc(producers=P, n_tokens=N, token_bytes=T, capacity=C, max_batch=mb)
        with hicr.Context(0, torch.cuda.current_stream().cuda_stream) as ctx:
            rings = [torch.zeros(T * C, dtype=torch.uint8, device="cuda") for _ in range(P)]
            srcs = [torch.from_numpy(cw.source_image(p)).cuda() for p in range(P)]
            sinks = [torch.zeros(N * T, dtype=torch.uint8, device="cuda") for _ in range(P)]
            rid, sid, kid = ([ctx.slot_register(t) for t in ts] for ts in (rings, srcs, sinks))
            m = ctx.mpsc_create(rid, T, C)
            m.stream(sid, kid, N, mb)
            torch.cuda.synchronize()
            assert all(torch.equal(a, b) for a, b in zip(srcs, sinks)), "mpsc sink"
            assert all(ctx.slot_counters(r) == (N, N) for r in rid)
    P, N, T, C = 4, 600, 32, 16
    tagged = W.generators.tagged_sources(P, N, T)
    with hicr.Context(0, torch.cuda.current_stream().cuda_stream) as ctx:
        ring = torch.zeros(T * C, dtype=torch.uint8, device="cuda")
        srcs = [torch.from_numpy(a).cuda() for a in tagged]
        sink = torch.zeros(P * N * T, dtype=torch.uint8, device="cuda")
        r = ctx.slot_register(ring)
        sid = [ctx.slot_register(t) for t in srcs]
        k = ctx.slot_register(sink)
        ch = ctx.channel_create(r, T, C)
        ch.locking_stream(sid, k, 0, N, 7)
        torch.cuda.synchronize()
        assert ch.counters() == (P * N, P * N) and ctx.slot_counters(k) == (0, P * N)

    # Global Memory Slots: put / get between two contexts, global fence
    gw = W.global_copy_graph(2)
    world, mem, oids, og = oracle_run(gw)
    ctxs = [hicr.Context(0, torch.cuda.current_stream().cuda_stream) for _ in range(2)]
    try:
        bufs = [{n: torch.from_numpy(gw.image(i, n)).cuda() for n in NAMES} for i in range(2)]
        ids = [{n: ctxs[i].slot_register(bufs[i][n]) for n in NAMES} for i in range(2)]
        gg = hicr.collective.exchange_in_process(ctxs, gw.tag, [[(2 * i, ids[i]["gsrc"]), (2 * i + 1, ids[i]["gdst"])] for i in range(2)])
        for i in range(2):
            ctxs[i].memcpy_batch(descs_for(gw, i, ids[i], gg[i]))
        hicr.collective.fence_in_process(ctxs)
        for i in range(2):
            for n in NAMES:
                assert bufs[i][n].cpu().numpy().tobytes() == mem[i][n].tobytes(), (i, n)
                assert ctxs[i].global_counters(ids[i][n]) == world.inst[i].slot_global_counters(oids[i][n])
    finally:
        for c in ctxs:
            c.close()
    print("sanitizer target ok: every kernel ran and matched the oracle")


if __name__ == "__main__":
    main()
