"""Randomised shapes through the device-resident channel runs (bulk-copy pipeline and vector
kernels alike): token size, capacity, producers, tokens, batch list and starting counters drawn
from a seed; sink, ring, head / tail and message counters against the oracle's call sequence."""
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


@pytest.mark.timeout(900)
@pytest.mark.parametrize("seed", range(24))
def test_random_mpsc_and_spsc_runs(hicr, seed, monkeypatch):
    if seed % 3 == 2:
        monkeypatch.setenv("HICR_PIPE_CLUSTER", "0")        # every third shape through the cooperative variant
    rng = np.random.default_rng(9000 + seed)
    T = int(rng.choice([16, 32, 48, 64, 80, 128, 256, 1024, 4096, 24, 7]))
    C = int(rng.choice([1, 2, 3, 8, 16, 48, 64, 100, 256, 1024]))
    P = int(rng.choice([1, 1, 2, 5, 17, 64, 148]))
    N = int(rng.integers(1, max(2, min(40000, (24 << 20) // (T * P)))))
    maxb = int(rng.integers(1, 2 * C + 2))
    pre = int(rng.integers(0, 2 * C + 1))
    o = Oracle()
    rings = [np.zeros(T * C, np.uint8) for _ in range(P)]
    srcs = [rng.integers(0, 256, (pre + N) * T, dtype=np.uint8) for _ in range(P)]
    sinks = [np.zeros((pre + N) * T, np.uint8) for _ in range(P)]
    rid = [o.slot_register(a) for a in rings]
    sid = [o.slot_register(a) for a in srcs]
    kid = [o.slot_register(a) for a in sinks]
    chs = [o.channel_create(rid[p], T, C)[1] for p in range(P)]

    def oracle_pushes(p, first, sizes):
        pos = first
        for b in sizes:
            left = int(b)
            while left:
                rc, k = o.channel_push(chs[p], sid[p], pos * T, left)
                assert rc == oracle.OK and k > 0
                assert o.channel_pop(chs[p], kid[p], pos * T, C) == (oracle.OK, k)
                pos += k
                left -= k

    with hicr.Context(0, torch.cuda.current_stream().cuda_stream) as ctx:
        g_r = [torch.from_numpy(a.copy()).cuda() for a in rings]
        g_s = [torch.from_numpy(a).cuda() for a in srcs]
        g_k = [torch.from_numpy(a.copy()).cuda() for a in sinks]
        assert [ctx.slot_register(t) for t in g_r + g_s + g_k] == rid + sid + kid
        if P == 1:
            ch = ctx.channel_create(rid[0], T, C)
            if pre:
                oracle_pushes(0, 0, [pre])
                ch.stream(sid[0], 0, kid[0], 0, [pre])
            sizes = W.generators._batches(rng, N, maxb)
            sizes = np.insert(sizes, int(rng.integers(0, len(sizes) + 1)), 0)          # a push of no tokens somewhere
            oracle_pushes(0, pre, sizes)
            ch.stream(sid[0], pre * T, kid[0], pre * T, sizes)
            assert ch.counters() == o.channel_counters(chs[0]) == (pre + N, pre + N)
        else:
            m = ctx.mpsc_create(rid, T, C)
            for first, count in ((0, pre), (pre, N)):
                if count == 0:
                    continue
                for p in range(P):
                    oracle_pushes(p, first, [maxb] * (count // maxb) + ([count % maxb] if count % maxb else []))
                m.stream(sid, kid, count, maxb, src_offs=[first * T] * P, dst_offs=[first * T] * P)
            for p in range(P):
                assert m.counters(p) == o.channel_counters(chs[p]) == (pre + N, pre + N)
        torch.cuda.synchronize()
        what = "seed %d: T=%d C=%d P=%d N=%d maxb=%d pre=%d" % (seed, T, C, P, N, maxb, pre)
        for p in range(P):
            assert g_k[p].cpu().numpy().tobytes() == sinks[p].tobytes(), what + " sink %d" % p
            assert g_r[p].cpu().numpy().tobytes() == rings[p].tobytes(), what + " ring %d" % p
        for s in rid + sid + kid:
            assert ctx.slot_counters(s) == o.slot_counters(s), what
