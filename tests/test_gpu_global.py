"""Parity of the Global Memory Slots on the CUDA path
against the oracle's World: the exchange (counts, lookup, duplicate keys), the three legal
directions and the rejected fourth, puts and gets between instances, every instance's memory
image, every slot's counters and the owner-side totals after the global fence -- bit-exact.

Instances are contexts.  Two set-ups: several contexts of this process on cuda:0 (the owner's
addresses are used as they are), and two PROCESSES on cuda:0 whose storage reaches each other
through CUDA IPC handles carried by a gloo group -- the path a one-process-per-GPU job takes over
NVLink.  (The pod has one GPU: the two processes' kernels never wait for each other -- each
fences locally, the count exchange runs on the host.)"""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle
import workloads as W
from global_common import NAMES, descs_for, oracle_run
from oracle.world import World
from parity import to_device_table

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

STATUS = {"ok": oracle.OK, "illegal_direction": oracle.ERR_ILLEGAL_DIRECTION, "duplicate_key": oracle.ERR_DUPLICATE_KEY,
          "out_of_bounds": oracle.ERR_OUT_OF_BOUNDS}


@pytest.fixture(scope="module")
def hicr():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import paper_2509_01425_b200 as h
    return h


def _instances(hicr, n):
    ctxs = [hicr.Context(0, torch.cuda.current_stream().cuda_stream) for _ in range(n)]
    for i, c in enumerate(ctxs):
        c.instance_set(i, n)
    return ctxs


def _close(ctxs):
    for c in ctxs:
        c.close()


def _bytes(s):
    return np.frombuffer(s.encode("ascii"), dtype=np.uint8).copy()


def _one(dst, dst_off, src, src_off, size):
    return W.make_descs([dst], [src], [dst_off], [src_off], [size])


def test_status_codes_match_the_oracle(hicr):
    assert hicr.HICR_ERR_ILLEGAL_DIRECTION == oracle.ERR_ILLEGAL_DIRECTION
    assert hicr.HICR_ERR_DUPLICATE_KEY == oracle.ERR_DUPLICATE_KEY


@pytest.mark.parametrize("device_table", [False, True])
def test_golden_directions_on_gpu(hicr, golden_dir, device_table):
    """The four slot-kind pairs: same verdict, same first bad
    index, same bytes and counters as the oracle, host- and device-validated."""
    cases = json.load(open(os.path.join(golden_dir, "global_examples.json")))["directions"]
    for c in cases:
        world = World(2)
        mem = [[np.full(32, 1 + 2 * i, np.uint8), np.full(32, 2 + 2 * i, np.uint8)] for i in range(2)]
        oid = [[world.inst[i].slot_register(a) for a in mem[i]] for i in range(2)]
        rc, og = world.exchange(7, [[(0, oid[0][1])], [(1, oid[1][1])]])
        assert rc == oracle.OK
        ctxs = _instances(hicr, 2)
        try:
            bufs = [[torch.from_numpy(a.copy()).cuda() for a in mem[i]] for i in range(2)]
            gid = [[ctxs[i].slot_register(t) for t in bufs[i]] for i in range(2)]
            assert gid == oid
            gg = hicr.collective.exchange_in_process(ctxs, 7, [[(0, gid[0][1])], [(1, gid[1][1])]])
            assert gg == og
            slot = {"L": gid[0][0], "G": gg[0][1]}
            dst, src = slot[c["dst"]], slot[c["src"]]
            if c["dst"] == c["src"] == "G":
                src = gg[0][0]
            if c["dst"] == c["src"] == "L":
                src = gid[0][1]
            d = np.concatenate([_one(gid[0][0], 0, gid[0][1], 0, 4), _one(dst, 4, src, 8, 16)])   # a valid one first
            orc, obad = world.inst[0].memcpy_batch(d)
            assert orc == STATUS[c["status"]], c["cite"]
            if device_table:
                t = torch.from_numpy(d.view(np.uint8).copy()).cuda()
                ctxs[0].memcpy_batch(t, n=len(d))
                if orc == oracle.OK:
                    ctxs[0].fence()
                else:
                    with pytest.raises(hicr.HicrError) as e:
                        ctxs[0].fence()
                    assert (e.value.status, e.value.first_bad) == (orc, obad), c["cite"]
            elif orc == oracle.OK:
                ctxs[0].memcpy_batch(d)
            else:
                with pytest.raises(hicr.HicrError) as e:
                    ctxs[0].memcpy_batch(d)
                assert (e.value.status, e.value.first_bad) == (orc, obad), c["cite"]
            world.fence_all()
            hicr.collective.fence_in_process(ctxs)
            for i in range(2):
                for a, t in zip(mem[i], bufs[i]):
                    assert t.cpu().numpy().tobytes() == a.tobytes(), c["cite"]          # rejected = no effect
                for s in list(gid[i]) + list(gg[i].values()):
                    assert ctxs[i].slot_counters(s) == world.inst[i].slot_counters(s), c["cite"]
                assert ctxs[i].global_counters(gid[i][1]) == world.inst[i].slot_global_counters(oid[i][1]), c["cite"]
        finally:
            _close(ctxs)


def test_golden_exchange_counts_lookup_and_duplicates(hicr, golden_dir):
    g = json.load(open(os.path.join(golden_dir, "global_examples.json")))
    for c in g["exchange"]:
        n = c["contributions"]
        ctxs = _instances(hicr, len(n))
        try:
            keep, contrib, key = [], [], 0
            for i, k in enumerate(n):
                mine = []
                for _ in range(k):
                    t = torch.zeros(8 + key, dtype=torch.uint8, device="cuda")
                    keep.append(t)
                    mine.append((key, ctxs[i].slot_register(t)))
                    key += 1
                contrib.append(mine)
            out = hicr.collective.exchange_in_process(ctxs, 7, contrib)
            for i in range(len(n)):
                assert len(out[i]) == c["received_by_each"] == sum(n), c["cite"]
                for k in range(sum(n)):
                    assert ctxs[i].global_lookup(7, k) == out[i][k]
                for bad in ((7, 99), (8, 0)):                                            # unknown key / unknown tag
                    with pytest.raises(hicr.HicrError) as e:
                        ctxs[i].global_lookup(*bad)
                    assert e.value.status == hicr.HICR_ERR_INVALID_SLOT
        finally:
            _close(ctxs)
    # duplicate keys: all-or-nothing, on every instance
    ctxs = _instances(hicr, 2)
    try:
        a, b = (torch.zeros(8, dtype=torch.uint8, device="cuda") for _ in range(2))
        sa, sb = ctxs[0].slot_register(a), ctxs[1].slot_register(b)
        with pytest.raises(hicr.HicrError) as e:
            hicr.collective.exchange_in_process(ctxs, 7, [[(0, sa)], [(0, sb)]])
        assert e.value.status == STATUS[g["duplicate_key"]["status"]], g["duplicate_key"]["cite"]
        with pytest.raises(hicr.HicrError):
            ctxs[0].global_lookup(7, 0)                                                  # nothing was created
        out = hicr.collective.exchange_in_process(ctxs, 7, [[(0, sa)], [(1, sb)]])
        hicr.collective.exchange_in_process(ctxs, 8, [[(0, sa)], [(1, sb)]])             # same keys, another tag
        with pytest.raises(hicr.HicrError) as e:
            hicr.collective.exchange_in_process(ctxs, 7, [[(1, sa)], []])                # (7, 1) exists
        assert e.value.status == hicr.HICR_ERR_DUPLICATE_KEY
        # only local slots are volunteered; a local slot behind a global one cannot be unregistered
        with pytest.raises(hicr.HicrError) as e:
            ctxs[0].global_volunteer(9, 5, out[0][1])
        assert e.value.status == hicr.HICR_ERR_INVALID_ARG
        with pytest.raises(hicr.HicrError) as e:
            ctxs[0].slot_unregister(sa)
        assert e.value.status == hicr.HICR_ERR_BUSY
        ctxs[0].slot_unregister(out[0][0])
        ctxs[0].slot_unregister(ctxs[0].global_lookup(8, 0))
        ctxs[0].slot_unregister(sa)
        with pytest.raises(hicr.HicrError):
            ctxs[0].global_lookup(7, 0)
    finally:
        _close(ctxs)


def test_golden_put_get_self_zero_oob_on_gpu(hicr, golden_dir):
    g = json.load(open(os.path.join(golden_dir, "global_examples.json")))
    ctxs = _instances(hicr, 2)
    try:
        bufs = [[torch.zeros(32, dtype=torch.uint8, device="cuda") for _ in range(2)] for _ in range(2)]
        ids = [[ctxs[i].slot_register(t) for t in bufs[i]] for i in range(2)]
        gg = hicr.collective.exchange_in_process(ctxs, 7, [[(0, ids[0][1])], [(1, ids[1][1])]])
        put = _bytes(g["put"]["payload"])
        bufs[0][0][:16] = torch.from_numpy(put).cuda()
        ctxs[0].memcpy_batch(_one(gg[0][1], 8, ids[0][0], 0, 16))
        hicr.collective.fence_in_process(ctxs)
        assert bufs[1][1][8:24].cpu().numpy().tobytes() == put.tobytes(), g["put"]["cite"]
        assert int(bufs[1][1][:8].sum()) == 0 and int(bufs[1][1][24:].sum()) == 0
        get = _bytes(g["get"]["payload"])
        bufs[1][1][:16] = torch.from_numpy(get).cuda()
        ctxs[0].memcpy_batch(_one(ids[0][0], 16, gg[0][1], 0, 16))
        hicr.collective.fence_in_process(ctxs)
        assert bufs[0][0][16:32].cpu().numpy().tobytes() == get.tobytes(), g["get"]["cite"]
        me = _bytes(g["self_get"]["payload"])
        bufs[0][1][:16] = torch.from_numpy(me).cuda()
        ctxs[0].memcpy_batch(_one(ids[0][0], 0, gg[0][0], 0, 16))
        hicr.collective.fence_in_process(ctxs)
        assert bufs[0][0][:16].cpu().numpy().tobytes() == me.tobytes(), g["self_get"]["cite"]
        before = [t.clone() for pair in bufs for t in pair]
        c0, g0 = ctxs[0].slot_counters(gg[0][1]), ctxs[1].global_counters(ids[1][1])
        ctxs[0].memcpy_batch(_one(gg[0][1], 32, ids[0][0], 32, 0))
        hicr.collective.fence_in_process(ctxs)
        assert all(torch.equal(a, b) for a, b in zip(before, [t for pair in bufs for t in pair])), g["zero_put"]["cite"]
        assert ctxs[0].slot_counters(gg[0][1]) == (c0[0], c0[1] + 1), g["zero_put"]["cite"]
        assert ctxs[1].global_counters(ids[1][1]) == (g0[0], g0[1] + 1), g["zero_put"]["cite"]
        with pytest.raises(hicr.HicrError) as e:
            ctxs[0].memcpy_batch(_one(ids[0][0], 0, gg[0][1], 20, 16))
        assert (e.value.status, e.value.first_bad) == (STATUS[g["oob_get"]["status"]], 0), g["oob_get"]["cite"]
    finally:
        _close(ctxs)


def test_rejected_batch_does_not_break_the_global_fence(hicr):
    """Instance 0's device table holds a put past the end of the peer's slot: the batch has no effect
    and the error surfaces at instance 0's half of the global fence -- after the count exchange, so
    instance 1's own put is fenced and counted as usual (oracle: same statuses, bytes and counts)."""
    world = World(2)
    mem = [[np.full(64, 1 + i, np.uint8), np.zeros(64, np.uint8)] for i in range(2)]
    oid = [[world.inst[i].slot_register(a) for a in mem[i]] for i in range(2)]
    rc, og = world.exchange(5, [[(0, oid[0][1])], [(1, oid[1][1])]])
    ctxs = _instances(hicr, 2)
    try:
        bufs = [[torch.from_numpy(a.copy()).cuda() for a in mem[i]] for i in range(2)]
        gid = [[ctxs[i].slot_register(t) for t in bufs[i]] for i in range(2)]
        gg = hicr.collective.exchange_in_process(ctxs, 5, [[(0, gid[0][1])], [(1, gid[1][1])]])
        bad = np.concatenate([_one(gg[0][1], 0, gid[0][0], 0, 16), _one(gg[0][1], 60, gid[0][0], 0, 16)])
        good = _one(gg[1][0], 8, gid[1][0], 0, 32)
        assert world.inst[0].memcpy_batch(bad) == (oracle.ERR_OUT_OF_BOUNDS, 1)
        assert world.inst[1].memcpy_batch(good)[0] == oracle.OK
        world.fence_all()
        t = torch.from_numpy(bad.view(np.uint8).copy()).cuda()
        ctxs[0].memcpy_batch(t, n=2)
        ctxs[1].memcpy_batch(good)
        with pytest.raises(hicr.HicrError) as e:
            hicr.collective.fence_in_process(ctxs)
        assert (e.value.status, e.value.first_bad) == (hicr.HICR_ERR_OUT_OF_BOUNDS, 1)
        for i in range(2):
            for a, tt in zip(mem[i], bufs[i]):
                assert tt.cpu().numpy().tobytes() == a.tobytes()
            for s_ in list(gid[i]) + list(gg[i].values()):
                assert ctxs[i].slot_counters(s_) == world.inst[i].slot_counters(s_)
            assert ctxs[i].global_counters(gid[i][1]) == world.inst[i].slot_global_counters(oid[i][1])
    finally:
        _close(ctxs)


def _compare_with_oracle(hicr, w, ctxs, bufs, ids, gg):
    world, mem, oids, og = oracle_run(w)
    assert ids == oids and gg == og
    for i in range(w.n_instances):
        for k in NAMES:
            assert bufs[i][k].cpu().numpy().tobytes() == mem[i][k].tobytes(), "instance %d %s" % (i, k)
        for s in list(ids[i].values()) + list(gg[i].values()):
            assert ctxs[i].slot_counters(s) == world.inst[i].slot_counters(s), "instance %d slot %d" % (i, s)
        for k in NAMES:
            assert ctxs[i].global_counters(ids[i][k]) == world.inst[i].slot_global_counters(oids[i][k]), (i, k)


@pytest.mark.parametrize("n_inst,device_tables,big", [(2, False, False), (3, True, False), (4, True, True), (2, False, True)])
def test_copy_graph_between_instances(hicr, n_inst, device_tables, big):
    """Random Local-to-Local / put / get transfers dealt to n instances, one global fence: every
    instance's four buffers, all per-slot counters and the owners' totals equal the oracle's.
    `big`: sizes up to 300 KB, so the chunk queue and the TMA path carry global slots too."""
    w = (W.global_copy_graph(n_inst, per_buffer=24, src_bytes=1 << 20, dst_bytes=8 << 20, max_size=300000, seed=W.BASE_SEED + 5)
         if big else W.global_copy_graph(n_inst))
    ctxs = _instances(hicr, n_inst)
    try:
        bufs = [{k: torch.from_numpy(w.image(i, k)).cuda() for k in NAMES} for i in range(n_inst)]
        ids = [{k: ctxs[i].slot_register(bufs[i][k]) for k in NAMES} for i in range(n_inst)]
        gg = hicr.collective.exchange_in_process(
            ctxs, w.tag, [[(2 * i, ids[i]["gsrc"]), (2 * i + 1, ids[i]["gdst"])] for i in range(n_inst)])
        keep = []
        for i in range(n_inst):
            d = descs_for(w, i, ids[i], gg[i])
            if device_tables:
                keep.append(torch.from_numpy(d.view(np.uint8).copy()).cuda())
                ctxs[i].memcpy_batch(keep[-1], n=len(d))
            else:
                ctxs[i].memcpy_batch(d)
        hicr.collective.fence_in_process(ctxs)
        _compare_with_oracle(hicr, w, ctxs, bufs, ids, gg)
    finally:
        _close(ctxs)


@pytest.mark.timeout(600)
def test_two_processes_over_cuda_ipc():
    """Two processes, one context each, on cuda:0; handles and fence counts travel over a gloo
    group; the storage of the other process is reached through CUDA IPC.  Each rank compares its
    own memory, counters and owner-side totals with the oracle's World (tests/global_two_proc.py
    exits non-zero on any difference)."""
    here = os.path.dirname(os.path.abspath(__file__))
    port = 29500 + os.getpid() % 2000
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, os.path.join(here, "global_two_proc.py")], env=dict(env, RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.STDOUT) for r in range(2)]
    outs = []
    for p in procs:
        try:
            out, _ = p.communicate(timeout=500)
        except subprocess.TimeoutExpired:
            p.kill()
            out, _ = p.communicate()
        outs.append(out.decode(errors="replace"))
    for r, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, "rank %d:\n%s" % (r, out[-3000:])
        assert "global two-process parity ok" in out


def test_recycled_index_starts_with_zero_owner_totals(hicr):
    """The owner-side totals belong to a registration, not to a table index: a slot registered at
    an index whose earlier slot had been volunteered starts at (0, 0), as the oracle's does
    (oracle_slot_register zeroes them), and the global fence waits for the NEW slot's transfers."""
    world = World(2)
    ctxs = _instances(hicr, 2)
    try:
        imgs = [np.zeros(4096, dtype=np.uint8), (np.arange(4096) % 251).astype(np.uint8)]
        o_imgs = [i.copy() for i in imgs]
        bufs = [torch.from_numpy(i).cuda() for i in imgs]
        sa, sb = ctxs[0].slot_register(bufs[0]), ctxs[1].slot_register(bufs[1])
        oa, ob = world.inst[0].slot_register(o_imgs[0]), world.inst[1].slot_register(o_imgs[1])
        out = hicr.collective.exchange_in_process(ctxs, 1, [[(0, sa)], []])
        rc, oout = world.exchange(1, [[(0, oa)], []])
        assert rc == oracle.OK
        put5 = lambda g, s: W.make_descs([g] * 5, [s] * 5, [0, 100, 200, 300, 400], [7, 9, 11, 13, 15], [64] * 5)
        ctxs[1].memcpy_batch(put5(out[1][0], sb))
        hicr.collective.fence_in_process(ctxs)
        assert world.inst[1].memcpy_batch(put5(oout[1][0], ob))[0] == oracle.OK
        world.fence_all()
        assert ctxs[0].global_counters(sa) == world.inst[0].slot_global_counters(oa) == (0, 5)
        # drop the global slot everywhere, then the local slot behind it; the index comes back
        for c, o in zip(ctxs, out):
            c.slot_unregister(o[0])
        ctxs[0].slot_unregister(sa)
        assert world.inst[0].slot_unregister(oa) == oracle.OK
        o_new = np.zeros(4096, dtype=np.uint8)
        new = torch.from_numpy(o_new.copy()).cuda()
        sa2, oa2 = ctxs[0].slot_register(new), world.inst[0].slot_register(o_new)
        assert sa2 != sa and (sa2 & 0xfff) == (sa & 0xfff)
        assert ctxs[0].global_counters(sa2) == world.inst[0].slot_global_counters(oa2) == (0, 0)
        out2 = hicr.collective.exchange_in_process(ctxs, 2, [[(0, sa2)], []])
        rc, oout2 = world.exchange(2, [[(0, oa2)], []])
        assert rc == oracle.OK
        two = lambda g, s: W.make_descs([g] * 2, [s] * 2, [5, 1000], [0, 2000], [333, 777])
        ctxs[1].memcpy_batch(two(out2[1][0], sb))
        hicr.collective.fence_in_process(ctxs)
        assert world.inst[1].memcpy_batch(two(oout2[1][0], ob))[0] == oracle.OK
        world.fence_all()
        assert ctxs[0].global_counters(sa2) == world.inst[0].slot_global_counters(oa2) == (0, 2)
        assert new.cpu().numpy().tobytes() == o_new.tobytes()
    finally:
        _close(ctxs)


def test_global_fence_keeps_the_error_with_more_than_64_global_slots(hicr):
    """hicr_global_fence_begin reports how much room it needs BEFORE it fences, so the retry with
    a larger array still returns the epoch's deferred error (66 global slots, one bad descriptor)."""
    ctxs = _instances(hicr, 2)
    try:
        bufs = [[torch.zeros(256, dtype=torch.uint8, device="cuda") for _ in range(33)] for _ in ctxs]
        ids = [[c.slot_register(b) for b in bb] for c, bb in zip(ctxs, bufs)]
        out = hicr.collective.exchange_in_process(ctxs, 3, [[(k, s) for k, s in enumerate(ids[0])],
                                                            [(100 + k, s) for k, s in enumerate(ids[1])]])
        assert len(out[0]) == 66
        bad = W.make_descs([out[0][100], out[0][101]], [ids[0][0], ids[0][1]], [0, 200], [0, 0], [16, 64])   # second: out of bounds
        t = to_device_table(bad)
        ctxs[0].memcpy_batch(t, n=2)
        with pytest.raises(hicr.HicrError) as e:
            hicr.collective.fence_in_process(ctxs)
        assert (e.value.status, e.value.first_bad) == (hicr.HICR_ERR_OUT_OF_BOUNDS, 1)
        assert ctxs[1].global_counters(ids[1][0]) == (0, 0)
        good = W.make_descs([out[0][100]], [ids[0][0]], [0], [0], [16])
        ctxs[0].memcpy_batch(good)
        hicr.collective.fence_in_process(ctxs)
        assert ctxs[1].global_counters(ids[1][0]) == (0, 1)
    finally:
        _close(ctxs)
