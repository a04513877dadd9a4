"""Pins for the CPU oracle's channel push / pop (CPU only).

Pinned against: the examples printed in SPEC (tests/golden/channel_examples.json), a
trivially correct queue of byte strings (collections.deque) under random schedules with
capacities 1..64, the closed forms of SURVEY.md S8(c) (head = tokens ever
pushed, tail = tokens ever popped, token i sits at ring offset (i mod C)*T, sink = source
prefix), and the invariants 0 <= head - tail <= C with monotone indices.
"""
import collections
import json
import os

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import Oracle


def _mk(T, C, src_tokens, sink_tokens, ring_fill=0xEE):
    o = Oracle()
    ring = np.full(T * C, ring_fill, dtype=np.uint8)
    src = np.zeros(max(1, src_tokens * T), dtype=np.uint8)
    sink = np.zeros(max(1, sink_tokens * T), dtype=np.uint8)
    r, s, k = o.slot_register(ring), o.slot_register(src), o.slot_register(sink)
    rc, ch = o.channel_create(r, T, C)
    assert rc == oracle.OK
    return o, ch, (ring, src, sink), (r, s, k)


def test_golden_channel_examples(golden_dir):
    cases = json.load(open(os.path.join(golden_dir, "channel_examples.json")))["cases"]
    assert len(cases) >= 4
    for c in cases:
        T, C = c["token_bytes"], c["capacity"]
        o, ch, (ring, src, sink), (r, s, k) = _mk(T, C, 8, 8)
        for op in c["ops"]:
            if op["op"] == "push":
                data = "".join(op["tokens"]).encode("ascii")
                src[: len(data)] = np.frombuffer(data, dtype=np.uint8)
                rc, n = o.channel_push(ch, s, 0, len(op["tokens"]))
            else:
                sink[:] = 0
                rc, n = o.channel_pop(ch, k, 0, op["max"])
                got = [sink[i * T: (i + 1) * T].tobytes().decode("ascii") for i in range(n)]
                assert got == op["popped"], c["cite"]
            assert rc == oracle.OK and n == op["returns"], c["cite"]
            h, t = o.channel_counters(ch)
            assert h - t == op["depth"], c["cite"]


def test_create_rejects_bad_configs():
    o = Oracle()
    ring = np.zeros(64, dtype=np.uint8)
    r = o.slot_register(ring)
    assert o.channel_create(r, 8, 0)[0] == oracle.ERR_INVALID_ARG       # capacity 0
    assert o.channel_create(r, 0, 8)[0] == oracle.ERR_INVALID_ARG
    assert o.channel_create(r, 8, 9)[0] == oracle.ERR_OUT_OF_BOUNDS     # ring slot too small
    assert o.channel_create(7, 8, 8)[0] == oracle.ERR_INVALID_SLOT
    assert o.channel_create(r, 8, 8)[0] == oracle.OK


@pytest.mark.parametrize("C", [1, 2, 3, 7, 16, 64])
@pytest.mark.parametrize("T", [1, 5, 64])
def test_differential_against_deque(C, T):
    """Random push/pop schedule; a deque of byte strings is the reference queue."""
    rng = np.random.default_rng(1000 * C + T)
    N = 4000
    o, ch, (ring, src, sink), (r, s, k) = _mk(T, C, N, N)
    src[:] = rng.integers(0, 256, src.size, dtype=np.uint8)
    q = collections.deque()
    pushed = popped = 0
    last_h = last_t = 0
    while popped < N:
        if pushed < N and rng.random() < 0.5:
            n = int(rng.integers(0, 2 * C + 2))
            n = min(n, N - pushed)
            rc, got = o.channel_push(ch, s, pushed * T, n)
            exp = min(n, C - len(q))
            assert rc == oracle.OK and got == exp                      # partial push (reading 12)
            for j in range(exp):
                q.append(src[(pushed + j) * T: (pushed + j + 1) * T].tobytes())
            pushed += exp
        else:
            m = int(rng.integers(0, 2 * C + 2))
            rc, got = o.channel_pop(ch, k, popped * T, m)
            exp = min(m, len(q))
            assert rc == oracle.OK and got == exp
            for j in range(exp):
                assert sink[(popped + j) * T: (popped + j + 1) * T].tobytes() == q.popleft()
            popped += exp
        h, t = o.channel_counters(ch)
        assert (h, t) == (pushed, popped)                               # closed form
        assert 0 <= h - t <= C and h >= last_h and t >= last_t
        assert h - t == len(q)
        last_h, last_t = h, t
        # token i (tail <= i < head) sits at ring offset (i mod C) * T
        for i in range(t, h):
            assert ring[(i % C) * T: (i % C + 1) * T].tobytes() == src[i * T: (i + 1) * T].tobytes()
    assert sink.tobytes() == src.tobytes()                              # FIFO, no loss, no dup
    # one message per token on the slot counters (reading 15)
    assert o.slot_counters(s) == (N, 0)
    assert o.slot_counters(r) == (N, N)
    assert o.slot_counters(k) == (0, N)


def test_push_pop_bounds():
    o, ch, (ring, src, sink), (r, s, k) = _mk(4, 4, 2, 2)
    assert o.channel_push(ch, s, 0, 3)[0] == oracle.ERR_OUT_OF_BOUNDS   # 12 bytes from an 8-byte slot
    assert o.channel_push(ch, 99, 0, 1)[0] == oracle.ERR_INVALID_SLOT
    assert o.channel_counters(ch) == (0, 0)
    assert o.channel_push(ch, s, 0, 2) == (oracle.OK, 2)
    assert o.channel_pop(ch, k, 4, 2)[0] == oracle.ERR_OUT_OF_BOUNDS    # 2 tokens at offset 4 of 8
    assert o.channel_counters(ch) == (2, 0)
    assert o.channel_pop(ch, k, 0, 2) == (oracle.OK, 2)


def test_config5a_schedule_scaled():
    """push(b_i) then pop(max = C): the ring is empty before every push, so every push
    returns b_i and every pop returns b_i (reading 13)."""
    w = W.spsc(n_tokens=20000, token_bytes=16, capacity=64, max_batch=64)
    T, C = w.token_bytes, w.capacity
    o, ch, (ring, src, sink), (r, s, k) = _mk(T, C, w.n_tokens, w.n_tokens)
    src[:] = w.source_image(0)
    pos = 0
    for b in w.batches[0]:
        assert o.channel_push(ch, s, pos * T, int(b)) == (oracle.OK, int(b))
        assert o.channel_pop(ch, k, pos * T, C) == (oracle.OK, int(b))
        pos += int(b)
    assert pos == w.n_tokens and o.channel_counters(ch) == (w.n_tokens, w.n_tokens)
    assert sink.tobytes() == src.tobytes()


def _run_mpsc(w, schedule):
    T, C, P, N = w.token_bytes, w.capacity, w.producers, w.n_tokens
    o = Oracle()
    rings = [np.zeros(T * C, dtype=np.uint8) for _ in range(P)]
    srcs = [w.source_image(p) for p in range(P)]
    sinks = [np.zeros(N * T, dtype=np.uint8) for _ in range(P)]
    rid = [o.slot_register(a) for a in rings]
    sid = [o.slot_register(a) for a in srcs]
    kid = [o.slot_register(a) for a in sinks]
    chs = [o.channel_create(rid[p], T, C)[1] for p in range(P)]
    nxt = [0] * P
    pushed = [0] * P
    popped = [0] * P
    for p in schedule:
        p = int(p)
        b = int(w.batches[p][nxt[p]])
        nxt[p] += 1
        done = 0
        while done < b:                          # blocking push = retry until room
            rc, k = o.channel_push(chs[p], sid[p], pushed[p] * T, b - done)
            assert rc == oracle.OK
            pushed[p] += k
            done += k
            rc, k = o.channel_pop(chs[p], kid[p], popped[p] * T, C)
            assert rc == oracle.OK
            popped[p] += k
    for p in range(P):
        assert o.channel_counters(chs[p]) == (N, N)
    return srcs, sinks


def test_mpsc_nonlocking_interleaving_independent():
    """Dedicated buffers per producer: per-producer FIFO, and the final
    image does not depend on the interleaving."""
    w = W.mpsc(producers=5, n_tokens=3000, token_bytes=8, capacity=32, max_batch=48)
    srcs, sinks = _run_mpsc(w, w.schedule)
    for a, b in zip(srcs, sinks):
        assert a.tobytes() == b.tobytes()
    other = np.random.default_rng(3).permutation(w.schedule)
    _, sinks2 = _run_mpsc(w, np.sort(other))     # producers strictly one after another
    for a, b in zip(sinks, sinks2):
        assert a.tobytes() == b.tobytes()


def test_mpsc_one_producer_equals_spsc():
    """producers = 1 -> behaviour equals SPSC."""
    w = W.mpsc(producers=1, n_tokens=2000, token_bytes=8, capacity=16, max_batch=16)
    srcs, sinks = _run_mpsc(w, w.schedule)
    assert srcs[0].tobytes() == sinks[0].tobytes()
