"""Parity of the channel path (hicr_channel_push / pop / stream, hicr_mpsc_stream; CUDA
through the C-ABI) against the CPU oracle: returned counts, head/tail, ring image, sink
image and slot message counters, bit-exact."""
import json
import os

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import Oracle

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def hicr():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import paper_2509_01425_b200 as h
    return h


def _ctx(hicr):
    return hicr.Context(0, torch.cuda.current_stream().cuda_stream)


def fence_counters_both(ctx, o, ids, what=""):
    """The kernels' own message counters (device memory), not the host mirror the channel calls
    keep: one zero-size descriptor (moves nothing, counts one message, reading 4) as a device
    batch + hicr_fence on the GPU, the same on the oracle, then every slot's counters.  The
    fence reads what the device counted (reading 15: one message per token)."""
    d = W.make_descs([ids[0]], [ids[-1]], [0], [0], [0])
    assert o.memcpy_batch(d)[0] == oracle.OK and o.fence() == oracle.OK
    t = torch.from_numpy(d.view(np.uint8).copy()).cuda()
    ctx.memcpy_batch(t, n=1)
    ctx.fence()
    for s in ids:
        assert ctx.slot_counters(s) == o.slot_counters(s), "%s device counters of slot %d" % (what, s)


class Pair:
    """The same ring / source / sink set up on the oracle and on the GPU."""

    def __init__(self, hicr, T, C, src_img, sink_bytes, ring_fill=0xEE):
        self.T, self.C = T, C
        self.o = Oracle()
        self.ring = np.full(T * C, ring_fill, dtype=np.uint8)
        self.src = src_img.copy()
        self.sink = np.zeros(sink_bytes, dtype=np.uint8)
        self.ids = [self.o.slot_register(a) for a in (self.ring, self.src, self.sink)]
        rc, self.och = self.o.channel_create(self.ids[0], T, C)
        assert rc == oracle.OK
        self.ctx = _ctx(hicr)
        self.g = [torch.from_numpy(a.copy()).cuda() for a in (self.ring, self.src, self.sink)]
        gids = [self.ctx.slot_register(t) for t in self.g]
        assert gids == self.ids
        self.ch = self.ctx.channel_create(gids[0], T, C)

    def check(self, what=""):
        torch.cuda.synchronize()
        assert self.ch.counters() == self.o.channel_counters(self.och), what
        for name, a, t in zip(("ring", "source", "sink"), (self.ring, self.src, self.sink), self.g):
            assert t.cpu().numpy().tobytes() == a.tobytes(), "%s %s differs" % (what, name)
        for s in self.ids:
            assert self.ctx.slot_counters(s) == self.o.slot_counters(s), "%s counters of slot %d" % (what, s)
        fence_counters_both(self.ctx, self.o, self.ids, what)

    def close(self):
        self.ctx.close()


def test_golden_channel_examples_on_gpu(hicr, golden_dir):
    cases = json.load(open(os.path.join(golden_dir, "channel_examples.json")))["cases"]
    for c in cases:
        T, C = c["token_bytes"], c["capacity"]
        with _ctx(hicr) as ctx:
            ring = torch.zeros(T * C, dtype=torch.uint8, device="cuda")
            src = torch.zeros(8 * T, dtype=torch.uint8, device="cuda")
            sink = torch.zeros(8 * T, dtype=torch.uint8, device="cuda")
            r, s, k = ctx.slot_register(ring), ctx.slot_register(src), ctx.slot_register(sink)
            ch = ctx.channel_create(r, T, C)
            for op in c["ops"]:
                if op["op"] == "push":
                    data = np.frombuffer("".join(op["tokens"]).encode("ascii"), dtype=np.uint8).copy()
                    src[: data.size] = torch.from_numpy(data).cuda()
                    n = ch.push(s, 0, len(op["tokens"]))
                else:
                    sink.zero_()
                    n = ch.pop(k, 0, op["max"])
                    out = sink.cpu().numpy()
                    assert [out[i * T: (i + 1) * T].tobytes().decode("ascii") for i in range(n)] == op["popped"], c["cite"]
                assert n == op["returns"], c["cite"]
                h, t = ch.counters()
                assert h - t == op["depth"], c["cite"]


def test_create_rejects_bad_configs(hicr):
    with _ctx(hicr) as ctx:
        ring = torch.zeros(64, dtype=torch.uint8, device="cuda")
        r = ctx.slot_register(ring)
        for (T, C, st) in [(8, 0, hicr.HICR_ERR_INVALID_ARG), (0, 8, hicr.HICR_ERR_INVALID_ARG),
                           (8, 9, hicr.HICR_ERR_OUT_OF_BOUNDS)]:
            with pytest.raises(hicr.HicrError) as e:
                ctx.channel_create(r, T, C)
            assert e.value.status == st
        with pytest.raises(hicr.HicrError) as e:
            ctx.channel_create(7, 8, 8)
        assert e.value.status == hicr.HICR_ERR_INVALID_SLOT
        ch = ctx.channel_create(r, 8, 8)
        with pytest.raises(hicr.HicrError) as e:
            ctx.slot_unregister(r)                      # ring still used by a live channel
        assert e.value.status == hicr.HICR_ERR_BUSY
        ch.close()
        ctx.slot_unregister(r)


@pytest.mark.parametrize("T,C", [(1, 1), (5, 3), (64, 7), (256, 16), (48, 64), (4096, 5), (33, 1024)])
def test_random_push_pop_schedule(hicr, T, C):
    """Random push / pop calls (including pushes into a full ring and pops from an empty
    one): every returned count and the final state equal the oracle's."""
    rng = np.random.default_rng(1000 + T * 7 + C)
    n_src = 6 * C + 40
    p = Pair(hicr, T, C, rng.integers(0, 256, n_src * T, dtype=np.uint8), n_src * T)
    try:
        pushed = popped = 0
        for step in range(120):
            if rng.random() < 0.55 and pushed < n_src:
                n = int(rng.integers(0, min(2 * C + 2, n_src - pushed) + 1))
                rc, k = p.o.channel_push(p.och, p.ids[1], pushed * T, n)
                assert rc == oracle.OK
                assert p.ch.push(p.ids[1], pushed * T, n) == k
                pushed += k
            else:
                m = int(rng.integers(0, 2 * C + 2))
                rc, k = p.o.channel_pop(p.och, p.ids[2], popped * T, m)
                assert rc == oracle.OK
                assert p.ch.pop(p.ids[2], popped * T, m) == k
                popped += k
            h, t = p.ch.counters()
            assert (h, t) == (pushed, popped) and 0 <= h - t <= C
        p.check("T=%d C=%d" % (T, C))
    finally:
        p.close()


def test_push_pop_bounds(hicr):
    T, C = 8, 4
    p = Pair(hicr, T, C, np.arange(64, dtype=np.uint8), 16)
    try:
        with pytest.raises(hicr.HicrError) as e:
            p.ch.push(p.ids[1], 0, 9)                    # 9 tokens = 72 B > 64 B source slot
        assert e.value.status == oracle.ERR_OUT_OF_BOUNDS == p.o.channel_push(p.och, p.ids[1], 0, 9)[0]
        assert p.ch.push(p.ids[1], 0, 4) == 4 == p.o.channel_push(p.och, p.ids[1], 0, 4)[1]
        with pytest.raises(hicr.HicrError) as e:
            p.ch.pop(p.ids[2], 0, 4)                     # 4 tokens = 32 B > 16 B sink: no effect
        assert e.value.status == oracle.ERR_OUT_OF_BOUNDS == p.o.channel_pop(p.och, p.ids[2], 0, 4)[0]
        assert p.ch.counters() == (4, 0)
        assert p.ch.pop(p.ids[2], 0, 2) == 2 == p.o.channel_pop(p.och, p.ids[2], 0, 2)[1]
        with pytest.raises(hicr.HicrError) as e:
            p.ch.push(99, 0, 1)
        assert e.value.status == oracle.ERR_INVALID_SLOT
        p.check()
    finally:
        p.close()


def _oracle_spsc(p, w):
    pos = 0
    for b in w.batches[0]:
        assert p.o.channel_push(p.och, p.ids[1], pos * p.T, int(b)) == (oracle.OK, int(b))
        assert p.o.channel_pop(p.och, p.ids[2], pos * p.T, p.C) == (oracle.OK, int(b))
        pos += int(b)


def test_config5a_host_calls_scaled(hicr):
    """Config 5a's loop -- push(b_i) then pop(max = C) -- through the host-call path."""
    w = W.spsc(n_tokens=30000, token_bytes=256, capacity=1024, max_batch=1024)
    p = Pair(hicr, w.token_bytes, w.capacity, w.source_image(0), w.n_tokens * w.token_bytes)
    try:
        _oracle_spsc(p, w)
        pos = 0
        for b in w.batches[0]:
            assert p.ch.push(p.ids[1], pos * p.T, int(b)) == int(b)
            assert p.ch.pop(p.ids[2], pos * p.T, p.C) == int(b)
            pos += int(b)
        p.check("5a host calls")
    finally:
        p.close()


@pytest.mark.parametrize("T,C,N,maxb", [(256, 1024, 200000, 1024), (7, 5, 3000, 9), (64, 1, 500, 3), (4096, 8, 4000, 32)])
def test_spsc_stream_equals_call_sequence(hicr, T, C, N, maxb):
    """hicr_channel_stream (device-resident producer and consumer in one kernel) leaves the
    sink, ring, head/tail and message counters exactly as the oracle's push/pop sequence."""
    w = W.spsc(n_tokens=N, token_bytes=T, capacity=C, max_batch=maxb)
    p = Pair(hicr, T, C, w.source_image(0), N * T)
    try:
        # the oracle drains fully after each push; blocking pushes larger than C are split
        pos = 0
        for b in w.batches[0]:
            left = int(b)
            while left:
                rc, k = p.o.channel_push(p.och, p.ids[1], pos * T, left)
                assert rc == oracle.OK and k > 0
                rc, k2 = p.o.channel_pop(p.och, p.ids[2], pos * T, C)
                assert k2 == k
                pos += k
                left -= k
        p.ch.stream(p.ids[1], 0, p.ids[2], 0, w.batches[0])
        p.check("stream T=%d C=%d" % (T, C))
        # and the channel is reusable by host calls afterwards, continuing the same counters
        assert p.ch.push(p.ids[1], 0, 1) == 1 == p.o.channel_push(p.och, p.ids[1], 0, 1)[1]
        assert p.ch.pop(p.ids[2], 0, 1) == 1 == p.o.channel_pop(p.och, p.ids[2], 0, 1)[1]
        p.check("after stream")
    finally:
        p.close()


@pytest.mark.parametrize("T,C,pre,batches", [
    (256, 1024, 37, [0, 5, 0, 3000, 1, 0, 1024, 2047, 0]),      # pushes of zero tokens, pushes larger than the ring
    (64, 48, 5, [100, 1, 1, 48, 49, 7]),                        # capacity not a power of two: pieces of 16 tokens
    (4096, 8, 3, [1, 30, 2, 9]),                                # two tokens per piece
    (16384, 4, 1, [5, 11]),                                     # a token larger than the default stage
    (1024, 1024, 77, [3000, 1, 2048, 700]),                     # a 1 MiB ring: four CTAs per end
    (32, 1024, 9, [4000, 96]),                                  # 1 KiB pieces: the smallest the pipeline takes
    (16, 64, 2, [500]),                                         # pieces below 1 KiB: the vector kernels
])
def test_stream_from_a_ring_in_use(hicr, T, C, pre, batches):
    """hicr_channel_stream on a channel whose counters are not at zero (host pushes / pops first, so
    the first piece starts inside a piece boundary), with the batch shapes above: sink, ring,
    head / tail and counters as the oracle's call sequence; then host calls again."""
    N = sum(batches)
    rng = np.random.default_rng(T + C)
    p = Pair(hicr, T, C, rng.integers(0, 256, (pre + N + 2) * T, dtype=np.uint8), (pre + N + 2) * T)
    try:
        for i in range(pre):                                     # one token in, one out: head = tail = pre
            assert p.ch.push(p.ids[1], i * T, 1) == 1 == p.o.channel_push(p.och, p.ids[1], i * T, 1)[1]
            assert p.ch.pop(p.ids[2], i * T, 1) == 1 == p.o.channel_pop(p.och, p.ids[2], i * T, 1)[1]
        pos = pre
        for b in batches:
            left = b
            while left:
                rc, k = p.o.channel_push(p.och, p.ids[1], pos * T, left)
                assert rc == oracle.OK and k > 0
                assert p.o.channel_pop(p.och, p.ids[2], pos * T, C) == (oracle.OK, k)
                pos += k
                left -= k
        p.ch.stream(p.ids[1], pre * T, p.ids[2], pre * T, batches)
        p.check("stream from head = tail = %d" % pre)
        assert p.ch.counters() == (pre + N, pre + N)
        assert p.ch.push(p.ids[1], pos * T, 2) == min(2, C) == p.o.channel_push(p.och, p.ids[1], pos * T, 2)[1]
        assert p.ch.pop(p.ids[2], pos * T, 2) == min(2, C) == p.o.channel_pop(p.och, p.ids[2], pos * T, 2)[1]
        p.check("after the run")
    finally:
        p.close()


@pytest.mark.parametrize("cluster", ["0", "1"])
def test_pipeline_with_and_without_clusters(hicr, monkeypatch, cluster):
    """HICR_PIPE_CLUSTER (read per call): the device-resident runs with the two ends of a ring as one
    thread-block cluster (default) and as two CTAs of a cooperative launch (the path for devices or
    shapes without clusters) -- the same results as the oracle either way."""
    monkeypatch.setenv("HICR_PIPE_CLUSTER", cluster)
    _mpsc_both(hicr, W.mpsc(producers=148, n_tokens=6000, token_bytes=64, capacity=1024, max_batch=256), 256)
    _mpsc_both(hicr, W.mpsc(producers=3, n_tokens=2000, token_bytes=48, capacity=64, max_batch=20), 20)
    T, C, N = 256, 1024, 100000
    w = W.spsc(n_tokens=N, token_bytes=T, capacity=C, max_batch=1024)
    p = Pair(hicr, T, C, w.source_image(0), N * T)
    try:
        _oracle_spsc(p, w)
        p.ch.stream(p.ids[1], 0, p.ids[2], 0, w.batches[0])
        p.check("spsc, HICR_PIPE_CLUSTER=" + cluster)
    finally:
        p.close()


def _mpsc_both(hicr, w, max_batch):
    T, C, P, N = w.token_bytes, w.capacity, w.producers, w.n_tokens
    # oracle: P independent SPSC channels driven in the seeded interleaving
    o = Oracle()
    rings = [np.zeros(T * C, dtype=np.uint8) for _ in range(P)]
    srcs = [w.source_image(p) for p in range(P)]
    sinks = [np.zeros(N * T, dtype=np.uint8) for _ in range(P)]
    rid = [o.slot_register(a) for a in rings]
    sid = [o.slot_register(a) for a in srcs]
    kid = [o.slot_register(a) for a in sinks]
    chs = [o.channel_create(rid[p], T, C)[1] for p in range(P)]
    nxt, pushed, popped = [0] * P, [0] * P, [0] * P
    for p in w.schedule:
        p = int(p)
        b = int(w.batches[p][nxt[p]])
        nxt[p] += 1
        done = 0
        while done < b:
            rc, k = o.channel_push(chs[p], sid[p], pushed[p] * T, b - done)
            pushed[p] += k
            done += k
            rc, k = o.channel_pop(chs[p], kid[p], popped[p] * T, C)
            popped[p] += k
    with _ctx(hicr) as ctx:
        g_r = [torch.from_numpy(a * 0).cuda() for a in rings]
        g_s = [torch.from_numpy(a).cuda() for a in srcs]
        g_k = [torch.zeros(N * T, dtype=torch.uint8, device="cuda") for _ in range(P)]
        assert [ctx.slot_register(t) for t in g_r] == rid
        assert [ctx.slot_register(t) for t in g_s] == sid
        assert [ctx.slot_register(t) for t in g_k] == kid
        m = ctx.mpsc_create(rid, T, C)
        m.stream(sid, kid, N, max_batch)
        torch.cuda.synchronize()
        for p in range(P):
            assert m.counters(p) == o.channel_counters(chs[p]) == (N, N)
            assert g_k[p].cpu().numpy().tobytes() == sinks[p].tobytes() == srcs[p].tobytes(), "sink %d" % p
            assert g_r[p].cpu().numpy().tobytes() == rings[p].tobytes(), "ring %d" % p
        for s in rid + sid + kid:
            assert ctx.slot_counters(s) == o.slot_counters(s)
        fence_counters_both(ctx, o, rid + sid + kid, "mpsc")


@pytest.mark.parametrize("P,N,T,C,maxb", [(1, 5000, 64, 16, 16), (5, 3000, 8, 32, 48), (148, 20000, 64, 1024, 256),
                                          (40, 1000, 100, 3, 7),
                                          (700, 600, 64, 64, 40)])     # more rings than fit the device at once: waves of clusters
def test_mpsc_stream(hicr, P, N, T, C, maxb):
    """Non-locking MPSC: one ring per producer, single consumer; per-producer
    sink = per-producer source, head_p = tail_p = N, independent of the interleaving."""
    w = W.mpsc(producers=P, n_tokens=N, token_bytes=T, capacity=C, max_batch=maxb)
    _mpsc_both(hicr, w, maxb)


@pytest.mark.parametrize("P,N1,N2,T,C,maxb", [(3, 1000, 777, 64, 48, 20), (148, 1500, 1100, 64, 1024, 256), (7, 10, 5, 24, 16, 3)])
def test_mpsc_stream_twice_continues_counters(hicr, P, N1, N2, T, C, maxb):
    """Two hicr_mpsc_stream runs on one channel set with N1 % C != 0: heads and tails keep
    counting (monotone indices), so the second run's first token goes to ring
    position N1 mod C, as the oracle's does.  Sources and sinks at non-zero offsets (the second
    run continues where the first stopped).  Ring images, head / tail, sinks and counters equal
    the oracle's after each run."""
    assert N1 % C != 0
    rng = np.random.default_rng(P * 131 + C)
    lead = 16 * int(rng.integers(1, 9))                    # sources start `lead` bytes into their slots
    srcs = [rng.integers(0, 256, lead + (N1 + N2) * T, dtype=np.uint8) for _ in range(P)]
    o = Oracle()
    rings = [np.zeros(T * C, dtype=np.uint8) for _ in range(P)]
    sinks = [np.zeros((N1 + N2) * T + 32, dtype=np.uint8) for _ in range(P)]
    rid = [o.slot_register(a) for a in rings]
    sid = [o.slot_register(a) for a in srcs]
    kid = [o.slot_register(a) for a in sinks]
    chs = [o.channel_create(rid[p], T, C)[1] for p in range(P)]

    def oracle_run(first, count):
        for p in range(P):
            done = 0
            while done < count:
                rc, k = o.channel_push(chs[p], sid[p], lead + (first + done) * T, min(count - done, maxb))
                assert rc == oracle.OK and k > 0
                assert o.channel_pop(chs[p], kid[p], 32 + (first + done) * T, C) == (oracle.OK, k)
                done += k

    with _ctx(hicr) as ctx:
        g_r = [torch.from_numpy(a.copy()).cuda() for a in rings]
        g_s = [torch.from_numpy(a).cuda() for a in srcs]
        g_k = [torch.from_numpy(a.copy()).cuda() for a in sinks]
        assert [ctx.slot_register(t) for t in g_r + g_s + g_k] == rid + sid + kid
        m = ctx.mpsc_create(rid, T, C)
        for first, count in ((0, N1), (N1, N2)):
            oracle_run(first, count)
            m.stream(sid, kid, count, maxb, src_offs=[lead + first * T] * P, dst_offs=[32 + first * T] * P)
            torch.cuda.synchronize()
            for p in range(P):
                assert m.counters(p) == o.channel_counters(chs[p]) == (first + count, first + count)
                assert g_k[p].cpu().numpy().tobytes() == sinks[p].tobytes(), "sink %d after %d" % (p, first + count)
                assert g_r[p].cpu().numpy().tobytes() == rings[p].tobytes(), "ring %d after %d" % (p, first + count)
            for s in rid + sid + kid:
                assert ctx.slot_counters(s) == o.slot_counters(s)
            fence_counters_both(ctx, o, rid + sid + kid, "mpsc run ending at %d" % (first + count))


def test_batch_then_channel_calls_then_fence(hicr):
    """memcpy_batch; channel_push / pop; fence on one context: the fence must report the batch's
    messages AND the channel's (the channel kernels count on the device after the batch's
    snapshot of the counters was taken).  Then the other order."""
    T, C = 32, 8
    rng = np.random.default_rng(5)
    p = Pair(hicr, T, C, rng.integers(0, 256, 40 * T, dtype=np.uint8), 40 * T)
    try:
        d = W.make_descs([p.ids[2]] * 3, [p.ids[1]] * 3, [600, 700, 800], [0, 64, 128], [64, 50, 1])
        t = torch.from_numpy(d.view(np.uint8).copy()).cuda()
        for order in (0, 1):
            if order == 0:
                assert p.o.memcpy_batch(d)[0] == oracle.OK
                p.ctx.memcpy_batch(t, n=len(d))
            for _ in range(3):
                assert p.ch.push(p.ids[1], 0, 5) == p.o.channel_push(p.och, p.ids[1], 0, 5)[1] == 5
                assert p.ch.pop(p.ids[2], 0, 8) == p.o.channel_pop(p.och, p.ids[2], 0, 8)[1] == 5
            if order == 1:
                assert p.o.memcpy_batch(d)[0] == oracle.OK
                p.ctx.memcpy_batch(t, n=len(d))
            assert p.o.fence() == oracle.OK
            p.ctx.fence()
            for s in p.ids:
                assert p.ctx.slot_counters(s) == p.o.slot_counters(s), "order %d slot %d" % (order, s)
        p.check("batch + channel + fence")
    finally:
        p.close()


# ------------------------------------------------------------ full-size configs 5a / 5b
@pytest.mark.timeout(1200)
def test_config5a_full_size_host_calls(hicr):
    """BASELINE.json config 5a exactly as worded -- "each push followed by a consumer pop of the
    available tokens" -- at FULL size (2^24 tokens of 256 B, capacity 1024, ~32.7 k batches)
    through hicr_channel_push / hicr_channel_pop, one launch per call: every returned count,
    then sink, ring, head / tail and message counters against the oracle's same call sequence."""
    w = W.spsc()
    assert w.n_tokens == 1 << 24 and w.token_bytes == 256 and w.capacity == 1024
    p = Pair(hicr, w.token_bytes, w.capacity, w.source_image(0), w.n_tokens * w.token_bytes)
    try:
        _oracle_spsc(p, w)
        pos = 0
        for b in w.batches[0]:
            b = int(b)
            assert p.ch.push(p.ids[1], pos * p.T, b) == b
            assert p.ch.pop(p.ids[2], pos * p.T, p.C) == b
            pos += b
        assert pos == 1 << 24 and p.ch.counters() == (1 << 24, 1 << 24)
        p.check("5a full size, host calls")
    finally:
        p.close()



@pytest.mark.timeout(900)
def test_config5a_full_size_stream(hicr):
    """BASELINE.json config 5a at FULL size (2^24 tokens of 256 B, capacity 1024, batches
    U{1..1024}) through the device-resident run bench.py times; the oracle does the push /
    pop(max = C) call sequence token by token.  Sink, ring, head/tail and message counters."""
    w = W.spsc()
    assert w.n_tokens == 1 << 24 and w.token_bytes == 256 and w.capacity == 1024
    p = Pair(hicr, w.token_bytes, w.capacity, w.source_image(0), w.n_tokens * w.token_bytes)
    try:
        pos = 0
        for b in w.batches[0]:
            b = int(b)
            assert p.o.channel_push(p.och, p.ids[1], pos * p.T, b) == (oracle.OK, b)
            assert p.o.channel_pop(p.och, p.ids[2], pos * p.T, p.C) == (oracle.OK, b)
            pos += b
        assert pos == 1 << 24
        p.ch.stream(p.ids[1], 0, p.ids[2], 0, w.batches[0])
        p.check("5a full size")
        assert p.ch.counters() == (1 << 24, 1 << 24)
    finally:
        p.close()


@pytest.mark.timeout(900)
def test_config5b_full_size_properties(hicr):
    """BASELINE.json config 5b at FULL size (148 producers x 2^20 tokens of 64 B): the result
    has a plain definition that needs no interleaving -- every sink equals its producer's
    source (per-producer FIFO), head_p = tail_p = 2^20, one message per token on every
    slot -- checked on the device for all 9.25 GiB."""
    w = W.mpsc()
    T, C, P, N = w.token_bytes, w.capacity, w.producers, w.n_tokens
    assert (P, N, T) == (148, 1 << 20, 64)
    with _ctx(hicr) as ctx:
        rings = [torch.zeros(T * C, dtype=torch.uint8, device="cuda") for _ in range(P)]
        srcs = [torch.from_numpy(w.source_image(p)).cuda() for p in range(P)]
        sinks = [torch.zeros(N * T, dtype=torch.uint8, device="cuda") for _ in range(P)]
        rid = [ctx.slot_register(t) for t in rings]
        sid = [ctx.slot_register(t) for t in srcs]
        kid = [ctx.slot_register(t) for t in sinks]
        m = ctx.mpsc_create(rid, T, C)
        m.stream(sid, kid, N, 256)
        torch.cuda.synchronize()
        for p in range(P):
            assert m.counters(p) == (N, N)
            assert torch.equal(sinks[p], srcs[p]), "sink %d" % p
            # the ring holds the last C tokens, token i at position i mod C (N is a multiple of C)
            assert torch.equal(rings[p], srcs[p][(N - C) * T:]), "ring %d" % p
            assert ctx.slot_counters(sid[p]) == (N, 0)
            assert ctx.slot_counters(rid[p]) == (N, N)
            assert ctx.slot_counters(kid[p]) == (0, N)


@pytest.mark.parametrize("s", [1, 7, 4096, (1 << 20) + 3])
def test_pingpong_capacity_one(hicr, s):
    """The paper's Test Case 1 shape: two opposing SPSC channels of capacity 1,
    one message of s bytes bounced A -> B -> A, several rounds; a second push before the pop
    returns 0 ("may not send any more messages").  Same buffers, rings, head /
    tail and slot counters as the oracle after every round."""
    rng = np.random.default_rng(s)
    imgs = [np.zeros(s, np.uint8), np.zeros(s, np.uint8), rng.integers(0, 256, s, dtype=np.uint8), np.zeros(s, np.uint8)]
    o = Oracle()
    oid = [o.slot_register(a) for a in imgs]
    oab, oba = o.channel_create(oid[0], s, 1)[1], o.channel_create(oid[1], s, 1)[1]
    with _ctx(hicr) as ctx:
        g = [torch.from_numpy(a.copy()).cuda() for a in imgs]
        ids = [ctx.slot_register(t) for t in g]
        assert ids == oid
        ab, ba = ctx.channel_create(ids[0], s, 1), ctx.channel_create(ids[1], s, 1)
        for r in range(3):
            assert ab.push(ids[2], 0, 1) == 1 == o.channel_push(oab, oid[2], 0, 1)[1]
            assert ab.push(ids[2], 0, 1) == 0 == o.channel_push(oab, oid[2], 0, 1)[1]      # full
            assert ab.pop(ids[3], 0, 1) == 1 == o.channel_pop(oab, oid[3], 0, 1)[1]
            assert ab.pop(ids[3], 0, 1) == 0 == o.channel_pop(oab, oid[3], 0, 1)[1]        # empty
            assert ba.push(ids[3], 0, 1) == 1 == o.channel_push(oba, oid[3], 0, 1)[1]
            assert ba.pop(ids[2], 0, 1) == 1 == o.channel_pop(oba, oid[2], 0, 1)[1]
            assert ab.counters() == o.channel_counters(oab) == (r + 1, r + 1)
            assert ba.counters() == o.channel_counters(oba) == (r + 1, r + 1)
        for t, a in zip(g, imgs):
            assert t.cpu().numpy().tobytes() == a.tobytes()
        assert imgs[3].tobytes() == imgs[2].tobytes()
        for i in ids:
            assert ctx.slot_counters(i) == o.slot_counters(i)
        fence_counters_both(ctx, o, ids, "ping-pong")


# ------------------------------------------------------------ locking MPSC
def _check_locking_sink(sink, srcs, T):
    """Invariants of a locking MPSC run, from the sink alone: every token is some producer's
    token (byte for byte), each producer's tokens appear in its own order, every token once."""
    P, N = len(srcs), srcs[0].size // T
    tok = sink.reshape(P * N, T)
    tag = np.ascontiguousarray(tok[:, :8]).view("<u4").reshape(P * N, 2)
    prod, idx = tag[:, 0].astype(np.int64), tag[:, 1].astype(np.int64)
    assert prod.min() >= 0 and prod.max() < P
    for p in range(P):
        mine = np.nonzero(prod == p)[0]
        assert mine.size == N, "producer %d: %d tokens in the sink" % (p, mine.size)
        assert np.array_equal(idx[mine], np.arange(N)), "producer %d out of order" % p       # FIFO, each once
        assert np.array_equal(tok[mine], srcs[p].reshape(N, T)), "producer %d payload" % p


@pytest.mark.timeout(600)
@pytest.mark.parametrize("P,N,T,C,maxb", [(1, 4000, 16, 8, 5), (4, 3000, 24, 16, 7), (37, 2000, 64, 64, 48),
                                          (148, 4096, 64, 1024, 256), (9, 500, 100, 1, 3)])
def test_mpsc_locking(hicr, P, N, T, C, maxb):
    """Locking MPSC: P producers share one ring through atomic reservation and
    in-order commit.  The interleaving is not defined, so the result is checked by its
    invariants; the same checker accepts the oracle's run of a seeded interleaving on one
    shared channel (sequential pushes = exclusive access), and head, tail and all message
    counters agree with it."""
    srcs = W.generators.tagged_sources(P, N, T)
    # oracle: one channel, producers take turns in a seeded order, consumer drains after each push
    o = Oracle()
    ring, sink = np.zeros(T * C, np.uint8), np.zeros(P * N * T, np.uint8)
    rid = o.slot_register(ring)
    sid = [o.slot_register(a.copy()) for a in srcs]
    kid = o.slot_register(sink)
    _, och = o.channel_create(rid, T, C)
    rng = np.random.default_rng(P * 1000 + C)
    left, pushed, popped = [N] * P, [0] * P, 0
    while any(left):
        p = int(rng.choice([q for q in range(P) if left[q]]))
        rc, k = o.channel_push(och, sid[p], pushed[p] * T, min(left[p], int(rng.integers(1, maxb + 1))))
        assert rc == oracle.OK and k > 0
        pushed[p] += k
        left[p] -= k
        rc, k2 = o.channel_pop(och, kid, popped * T, C)
        assert k2 == k
        popped += k
    _check_locking_sink(sink, srcs, T)

    with _ctx(hicr) as ctx:
        g_ring = torch.zeros(T * C, dtype=torch.uint8, device="cuda")
        g_src = [torch.from_numpy(a).cuda() for a in srcs]
        g_sink = torch.zeros(P * N * T, dtype=torch.uint8, device="cuda")
        assert ctx.slot_register(g_ring) == rid
        assert [ctx.slot_register(t) for t in g_src] == sid
        assert ctx.slot_register(g_sink) == kid
        ch = ctx.channel_create(rid, T, C)
        ch.locking_stream(sid, kid, 0, N, maxb)
        torch.cuda.synchronize()
        _check_locking_sink(g_sink.cpu().numpy(), srcs, T)
        assert ch.counters() == o.channel_counters(och) == (P * N, P * N)
        for s in [rid, kid] + sid:
            assert ctx.slot_counters(s) == o.slot_counters(s)
        fence_counters_both(ctx, o, [rid, kid] + sid, "locking mpsc")
        # the channel keeps working through host calls afterwards, on the same counters
        assert ch.push(sid[0], 0, 1) == 1 and ch.pop(kid, 0, 1) == 1
        assert ch.counters() == (P * N + 1, P * N + 1)
