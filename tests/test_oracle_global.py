"""Pins for the oracle's Global Memory Slots (CPU only, -m "not gpu").

PAPER.md:377-383 (S3.1.4): the collective exchange, "uniquely identified by a tag and key pair",
the three legal directions, "Global-to-Global operations are not permitted".  The oracle
(hicr_oracle.c + world.py) is pinned against the examples the SPEC prints (tests/golden/
global_examples.json, each with its citation), against numpy slicing on a flat model of all
instances' memories under a randomized copy graph, and against closed-form counts.
"""
import json
import os

import numpy as np
import pytest

import oracle
import workloads as W
from oracle.world import World

STATUS = {"ok": oracle.OK, "illegal_direction": oracle.ERR_ILLEGAL_DIRECTION, "duplicate_key": oracle.ERR_DUPLICATE_KEY,
          "out_of_bounds": oracle.ERR_OUT_OF_BOUNDS}


def _bytes(s):
    return np.frombuffer(s.encode("ascii"), dtype=np.uint8).copy()


def _one(dst, dst_off, src, src_off, size):
    return W.make_descs([dst], [src], [dst_off], [src_off], [size])


@pytest.fixture(scope="module")
def golden(golden_dir):
    return json.load(open(os.path.join(golden_dir, "global_examples.json")))


def _two_instances():
    """Instances 0 and 1, each with a local buffer and one volunteered slot (keys 0 and 1, tag 7)."""
    w = World(2)
    mem = [[np.zeros(32, np.uint8), np.zeros(32, np.uint8)] for _ in range(2)]      # [instance][local, volunteered]
    ids = [[w.inst[i].slot_register(a) for a in mem[i]] for i in range(2)]
    rc, g = w.exchange(7, [[(0, ids[0][1])], [(1, ids[1][1])]])
    assert rc == oracle.OK
    return w, mem, ids, g


def test_golden_directions(golden):
    """Exactly the (global, global) pair is rejected, the other three are carried out."""
    assert len(golden["directions"]) == 4
    for c in golden["directions"]:
        w, mem, ids, g = _two_instances()
        mem[0][0][:] = 1
        mem[0][1][:] = 2
        mem[1][1][:] = 3
        # instance 0 initiates; L = its local buffer, G = a global slot (the peer's for one side,
        # its own for the other when both are global)
        slot = {"L": ids[0][0], "G": g[0][1]}
        dst, src = slot[c["dst"]], slot[c["src"]]
        if c["dst"] == c["src"] == "G":
            src = g[0][0]
        if c["dst"] == c["src"] == "L":
            src = ids[0][1]
        rc, bad = w.inst[0].memcpy_batch(_one(dst, 4, src, 8, 16))
        assert rc == STATUS[c["status"]], c["cite"]
        if rc != oracle.OK:
            assert bad == 0
            assert all((a == v).all() for a, v in ((mem[0][0], 1), (mem[0][1], 2), (mem[1][1], 3))), "rejected = no effect"
        w.fence_all()
        total = sum(sum(w.inst[i].slot_counters(s)) for i in range(2) for s in range(4))
        assert total == (2 if rc == oracle.OK else 0), c["cite"]


def test_golden_exchange_counts(golden):
    """"returns as many global memory slots as the total amount of local memory slots exchanged"
    (PAPER.md:379): every instance receives sum(contributions) slots, and all agree on the keys."""
    for c in golden["exchange"]:
        n = c["contributions"]
        w = World(len(n))
        contrib, key = [], 0
        for i, k in enumerate(n):
            mine = []
            for _ in range(k):
                mine.append((key, w.inst[i].slot_register(np.zeros(8 + key, np.uint8))))
                key += 1
            contrib.append(mine)
        rc, out = w.exchange(7, contrib)
        assert rc == oracle.OK, c["cite"]
        assert sum(n) == c["received_by_each"], c["cite"]
        for i in range(len(n)):
            assert len(out[i]) == c["received_by_each"], c["cite"]
            assert sorted(out[i]) == list(range(sum(n))), c["cite"]              # same key set everywhere
            for k in range(sum(n)):
                assert w.lookup(i, 7, k) == out[i][k]                              # getGlobalSlot
        assert w.lookup(0, 7, 99) is None and w.lookup(0, 8, 0) is None             # unknown key / unknown tag


def test_golden_duplicate_key(golden):
    c = golden["duplicate_key"]
    w = World(2)
    a, b = w.inst[0].slot_register(np.zeros(8, np.uint8)), w.inst[1].slot_register(np.zeros(8, np.uint8))
    rc, out = w.exchange(7, [[(0, a)], [(0, b)]])
    assert rc == STATUS[c["status"]] and out is None, c["cite"]
    assert w.lookup(0, 7, 0) is None, "a failed exchange creates nothing"
    # the same keys under another tag are fine, and a second exchange may not reuse (tag, key)
    assert w.exchange(7, [[(0, a)], [(1, b)]])[0] == oracle.OK
    assert w.exchange(8, [[(0, a)], [(1, b)]])[0] == oracle.OK
    assert w.exchange(7, [[(1, a)], []])[0] == oracle.ERR_DUPLICATE_KEY


def test_golden_put_get_self_zero_oob(golden):
    w, mem, ids, g = _two_instances()
    # put: instance 0 writes its local bytes into instance 1's volunteered slot
    p = _bytes(golden["put"]["payload"])
    mem[0][0][:16] = p
    assert w.inst[0].memcpy_batch(_one(g[0][1], 8, ids[0][0], 0, 16))[0] == oracle.OK
    w.fence_all()
    assert mem[1][1][8:24].tobytes() == p.tobytes(), golden["put"]["cite"]
    assert mem[1][1][:8].sum() == 0 and mem[1][1][24:].sum() == 0
    # get: instance 0 reads what instance 1 holds
    q = _bytes(golden["get"]["payload"])
    mem[1][1][:16] = q
    assert w.inst[0].memcpy_batch(_one(ids[0][0], 16, g[0][1], 0, 16))[0] == oracle.OK
    w.fence_all()
    assert mem[0][0][16:32].tobytes() == q.tobytes(), golden["get"]["cite"]
    # self-loop: a get from the instance's own global slot is a local copy
    s = _bytes(golden["self_get"]["payload"])
    mem[0][1][:16] = s
    assert w.inst[0].memcpy_batch(_one(ids[0][0], 0, g[0][0], 0, 16))[0] == oracle.OK
    w.fence_all()
    assert mem[0][0][:16].tobytes() == s.tobytes(), golden["self_get"]["cite"]
    # zero-size put: counters advance, no bytes move
    before = [m.copy() for pair in mem for m in pair]
    c0 = w.inst[0].slot_counters(g[0][1])
    gc0 = w.inst[1].slot_global_counters(ids[1][1])
    assert w.inst[0].memcpy_batch(_one(g[0][1], 32, ids[0][0], 32, 0))[0] == oracle.OK
    w.fence_all()
    assert [m.tobytes() for pair in mem for m in pair] == [m.tobytes() for m in before], golden["zero_put"]["cite"]
    assert w.inst[0].slot_counters(g[0][1]) == (c0[0], c0[1] + 1), golden["zero_put"]["cite"]
    assert w.inst[1].slot_global_counters(ids[1][1]) == (gc0[0], gc0[1] + 1), golden["zero_put"]["cite"]
    # out of bounds on the remote side rejects the batch
    rc, bad = w.inst[0].memcpy_batch(_one(ids[0][0], 0, g[0][1], 20, 16))
    assert rc == STATUS[golden["oob_get"]["status"]] and bad == 0, golden["oob_get"]["cite"]


def test_global_slot_is_the_owners_storage():
    """A Global Memory Slot has the size and the bytes of the local slot behind it, on every
    instance ("local memory slots that are made accessible to other HiCR instances")."""
    w, mem, ids, g = _two_instances()
    mem[1][1][:] = np.arange(32, dtype=np.uint8)
    for i in range(2):
        dst = np.zeros(32, np.uint8)
        d = w.inst[i].slot_register(dst)
        assert w.inst[i].memcpy_batch(_one(d, 0, g[i][1], 0, 32))[0] == oracle.OK       # whole slot: exact fit
        assert w.inst[i].memcpy_batch(_one(d, 0, g[i][1], 0, 33))[0] == oracle.ERR_OUT_OF_BOUNDS
        assert dst.tobytes() == mem[1][1].tobytes()
    # only local slots are volunteered
    assert w.exchange(9, [[(5, g[0][1])], []])[0] == oracle.ERR_INVALID_ARG
    assert w.exchange(9, [[(5, 99)], []])[0] == oracle.ERR_INVALID_SLOT
    rc, _ = w.inst[0].slot_register_global(w.inst[0], g[0][1])
    assert rc == oracle.ERR_INVALID_ARG


@pytest.mark.parametrize("seed", range(6))
def test_random_copy_graph_matches_numpy_model(seed):
    """SPEC.md:306 "randomized copy-graph property test": n instances, local and global slots,
    random legal transfers under the epoch precondition (destinations pairwise disjoint over ALL
    instances, no destination overlapping a source), one global fence.  The model is numpy
    slicing on snapshots: out[x] = before[src_off + x - dst_off]; counters are np.bincount."""
    rng = np.random.default_rng(500 + seed)
    n_inst = int(rng.integers(2, 5))
    w = World(n_inst)
    SRC, DST = 256, 1024
    # per instance: a private local source, a private local destination, a volunteered source and a
    # volunteered destination (sources are only read, destinations only written: the precondition holds)
    mem = [{k: rng.integers(0, 256, SRC if k.endswith("src") else DST, dtype=np.uint8)
            for k in ("lsrc", "ldst", "gsrc", "gdst")} for _ in range(n_inst)]
    ids = [{k: w.inst[i].slot_register(a) for k, a in mem[i].items()} for i in range(n_inst)]
    rc, g = w.exchange(3, [[(2 * i, ids[i]["gsrc"]), (2 * i + 1, ids[i]["gdst"])] for i in range(n_inst)])
    assert rc == oracle.OK
    before = [{k: a.copy() for k, a in m.items()} for m in mem]
    expect = [{k: a.copy() for k, a in m.items()} for m in mem]
    # destination ranges: disjoint pieces of every destination buffer, dealt to random initiators
    plans = [[] for _ in range(n_inst)]
    own = np.zeros((n_inst, 8), dtype=np.int64)          # [instance][slot id] -> (sent, recv) closed form
    cnt = [dict() for _ in range(n_inst)]
    gcnt = {}
    for owner in range(n_inst):
        for kind in ("ldst", "gdst"):
            sizes = rng.integers(0, 40, size=12)
            offs = W.gaps_composition(rng, sizes, 0, DST)
            for sz, off in zip(sizes, offs):
                sz, off = int(sz), int(off)
                if kind == "ldst":
                    init = owner                                      # a local slot is reachable by its instance only
                    dst_id = ids[owner]["ldst"]
                    src_owner = int(rng.integers(0, n_inst))
                    if src_owner == init and rng.random() < 0.5:
                        src_kind, src_id = "lsrc", ids[init]["lsrc"]                  # Local-to-Local
                    else:
                        src_kind, src_id = "gsrc", g[init][2 * src_owner]             # Global-to-Local (get)
                else:
                    init = int(rng.integers(0, n_inst))                               # Local-to-Global (put)
                    dst_id = g[init][2 * owner + 1]
                    src_owner, src_kind, src_id = init, "lsrc", ids[init]["lsrc"]
                so = int(rng.integers(0, SRC - sz + 1))
                plans[init].append((dst_id, off, src_id, so, sz))
                expect[owner][kind][off:off + sz] = before[src_owner][src_kind][so:so + sz]
                for (inst, sid, col) in ((init, src_id, 0), (init, dst_id, 1)):
                    c = cnt[inst].setdefault(sid, [0, 0])
                    c[col] += 1
                if src_kind == "gsrc":
                    gcnt.setdefault((src_owner, ids[src_owner]["gsrc"]), [0, 0])[0] += 1
                if kind == "gdst":
                    gcnt.setdefault((owner, ids[owner]["gdst"]), [0, 0])[1] += 1
    for i in rng.permutation(n_inst):                                                 # any instance order
        p = plans[int(i)]
        order = rng.permutation(len(p))
        d = W.make_descs(*[[p[j][c] for j in order] for c in (0, 2, 1, 3, 4)])
        assert w.inst[int(i)].memcpy_batch(d)[0] == oracle.OK
    assert w.fence_all() == [oracle.OK] * n_inst
    for i in range(n_inst):
        for k in mem[i]:
            assert mem[i][k].tobytes() == expect[i][k].tobytes(), "instance %d %s" % (i, k)
        n_ids = 4 + 2 * n_inst
        for sid in range(n_ids):
            assert list(w.inst[i].slot_counters(sid)) == cnt[i].get(sid, [0, 0]), "instance %d slot %d" % (i, sid)
        for k in ("lsrc", "ldst", "gsrc", "gdst"):
            assert list(w.inst[i].slot_global_counters(ids[i][k])) == gcnt.get((i, ids[i][k]), [0, 0])
    # the owner's global counters = the sum over instances of their own counts on that global slot
    for owner in range(n_inst):
        for key, name in ((2 * owner, "gsrc"), (2 * owner + 1, "gdst")):
            tot = np.sum([w.inst[i].slot_counters(g[i][key]) for i in range(n_inst)], axis=0)
            assert tuple(int(x) for x in tot) == w.inst[owner].slot_global_counters(ids[owner][name])
