"""Parity of hicr_memcpy_batch / hicr_fence (CUDA, through the C-ABI) against the CPU oracle.

Bit-exact: the path is pure data movement, so every destination byte, every byte outside
the destination ranges and every counter must equal the oracle's (north_star (d)).
"""
import json
import os

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import Oracle
from parity import assert_same, run_gpu, run_oracle, to_device_table

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


def _bytes(s):
    return np.frombuffer(s.encode("ascii"), dtype=np.uint8).copy()


# ------------------------------------------------------------------ printed examples
def test_golden_examples_on_gpu(hicr, golden_dir):
    """The SPEC/paper printed examples (tests/golden/memcpy_examples.json), through CUDA."""
    status = {"ok": hicr.HICR_OK, "out_of_bounds": hicr.HICR_ERR_OUT_OF_BOUNDS, "invalid_slot": hicr.HICR_ERR_INVALID_SLOT}
    cases = json.load(open(os.path.join(golden_dir, "memcpy_examples.json")))["cases"]
    for c in cases:
        m = c["memcpy"]
        overlapping = m["dst"] == m["src"] and m["size"] and \
            m["dst_off"] < m["src_off"] + m["size"] and m["src_off"] < m["dst_off"] + m["size"]
        if overlapping:
            continue  # a self-overlapping copy violates the epoch precondition (reading 5)
        with _ctx(hicr) as ctx:
            bufs = [torch.from_numpy(_bytes(s)).cuda() if len(s) else torch.empty(0, dtype=torch.uint8, device="cuda")
                    for s in c["slots"]]
            ids = [ctx.slot_register(b) for b in bufs]
            d = W.make_descs([ids[m["dst"]]], [ids[m["src"]]], [m["dst_off"]], [m["src_off"]], [m["size"]])
            rc = hicr.HICR_OK
            try:
                ctx.memcpy_batch(d)
            except hicr.HicrError as e:
                rc = e.status
                assert e.first_bad == 0
            assert rc == status[c["status"]], c["cite"]
            ctx.fence()
            for b, e in zip(bufs, c["expect"]):
                assert b.cpu().numpy().tobytes().decode("ascii") == e, c["cite"]


def test_broadcast_listing_on_gpu(hicr, golden_dir):
    """one message into N fresh slots at offset 0, a single fence."""
    g = json.load(open(os.path.join(golden_dir, "broadcast.json")))
    msg = _bytes(g["message"])
    rng = np.random.default_rng(7)
    dsts = [rng.integers(0, 256, g["destination_size"], dtype=np.uint8) for _ in range(g["n_destinations"])]
    with _ctx(hicr) as ctx:
        m = ctx.slot_register(torch.from_numpy(msg).cuda())
        bufs = [torch.from_numpy(d).cuda() for d in dsts]
        ids = [ctx.slot_register(b) for b in bufs]
        for i in ids:
            ctx.memcpy_batch(W.make_descs([i], [m], [0], [0], [msg.size]))
        ctx.fence()
        for b, d in zip(bufs, dsts):
            out = b.cpu().numpy()
            assert out[: msg.size].tobytes() == msg.tobytes()
            assert out[msg.size:].tobytes() == d[msg.size:].tobytes()
        assert ctx.slot_counters(m) == (len(ids), 0)
        assert all(ctx.slot_counters(i) == (0, 1) for i in ids)


# ------------------------------------------------- every alignment x ragged sizes
SIZES = [0, 1, 2, 3, 15, 16, 17, 31, 32, 33, 47, 48, 63, 64, 65, 127, 128, 129, 255, 256, 257, 500, 511, 512, 513,
         1023, 1024, 1025, 4095, 4096, 4097, 8191, 8192, 8193, 12345, 32767, 32768, 32769, 65535, 65536, 65537,
         100003, 262144 + 5]


def _alignment_workload(sizes, seed):
    """Every (dst mod 16, src mod 16) pair for every size in ``sizes``: destinations laid
    end to end with the wanted alignment in slot 1, sources at the wanted alignment in slot 0."""
    rng = np.random.default_rng(seed)
    dst_off, src_off, size = [], [], []
    pos = 0
    max_size = max(sizes)
    src_bytes = max_size + 4096
    for n in sizes:
        for da in range(16):
            for sa in range(16):
                pos = (pos + 15) // 16 * 16 + da + 16 * int(rng.integers(0, 3))
                dst_off.append(pos)
                pos += n
                s = int(rng.integers(0, (src_bytes - n - 16) // 16)) * 16 + sa
                src_off.append(s)
                size.append(n)
    d = W.make_descs(1, 0, dst_off, src_off, size)
    d = d[rng.permutation(len(d))]
    w = W.CopyWorkload("alignment", 1, [src_bytes, pos + 64], [d], seed=seed)
    return w


@pytest.mark.parametrize("group", [0, 1, 2])
@pytest.mark.parametrize("device_tables", [False, True])
def test_every_alignment_and_ragged_size(hicr, group, device_tables):
    """Brute force over head/body/tail handling: 256 alignment pairs x sizes that span the
    byte head, the 16 B vector body (aligned and byte-shifted loads), ragged last tiles,
    the warp-queue / chunk-queue boundary and multi-chunk descriptors."""
    sizes = SIZES[group::3]
    w = _alignment_workload(sizes, seed=100 + group)
    from oracle import hazard
    assert hazard.check(w.epochs[0], w.slot_sizes) is None
    assert_same(w, run_oracle(w), run_gpu(w, device_tables=device_tables), "group %d" % group)


def test_same_slot_source_and_destination(hicr):
    """src and dst in the same slot, disjoint ranges, odd alignments (config 4's shape)."""
    w = W.chained_epochs(n_epochs=1, n_desc=4096, slot_bytes=4 * W.MiB, smin=1, smax=700)
    assert_same(w, run_oracle(w), run_gpu(w))


# ------------------------------------------------------------- scaled configs 1-4
SMALL = {
    "tiny": lambda: W.tiny(),
    "bulk": lambda: W.bulk_aligned(n_desc=2048, slot_bytes=64 * W.MiB, n_sets=4),
    "heavy_a": lambda: W.heavy_tailed("a", n_slots=8, slot_bytes=16 * W.MiB, src_zone=2 * W.MiB,
                                      n_desc=3000, smax=2 * W.MiB),
    "heavy_b": lambda: W.heavy_tailed("b", n_slots=8, slot_bytes=16 * W.MiB, src_zone=2 * W.MiB,
                                      n_desc=6000, smax=2 * W.MiB),
    "chain": lambda: W.chained_epochs(n_epochs=8, n_desc=8192, slot_bytes=8 * W.MiB),
}


@pytest.mark.parametrize("name", sorted(SMALL))
@pytest.mark.parametrize("device_tables", [False, True])
def test_scaled_configs(hicr, name, device_tables):
    w = SMALL[name]()
    ref = run_oracle(w)
    assert_same(w, ref, run_gpu(w, device_tables=device_tables))


@pytest.mark.parametrize("name", ["tiny", "heavy_a"])
def test_several_batches_one_fence(hicr, name):
    """An epoch submitted as 7 batches before its single fence (the paper's listing issues
    one memcpy per destination, then one fence) equals one batch.  More
    batches than internal control blocks are covered by split=100."""
    w = SMALL[name]()
    ref = run_oracle(w)
    assert_same(w, ref, run_gpu(w, split=7))
    assert_same(w, ref, run_gpu(w, split=100, device_tables=True))


@pytest.mark.parametrize("name", ["tiny", "chain"])
def test_host_tables_split_epochs(hicr, name):
    """Configs 1 and 4 with every epoch cut into several HOST-table batches before its fence."""
    w = SMALL[name]()
    ref = run_oracle(w)
    assert_same(w, ref, run_gpu(w, split=3))
    assert_same(w, ref, run_gpu(w, split=9))


def test_more_host_batches_than_completion_records(hicr):
    """One epoch of 150 HOST-table batches of mixed sizes, among them tables of more than 1 MiB
    between short ones (a short table is read from pinned staging in place, a long one is
    copied): the epoch drains its 64 completion records twice while staging blocks are in use,
    and no block may be recycled before the kernel that reads it has run."""
    w = W.bulk_aligned(n_desc=150000, slot_bytes=256 * W.MiB, page=256, n_sets=1)
    ref = run_oracle(w)
    d = w.epochs[0]
    rng = np.random.default_rng(11)
    cuts, pos = [], 0
    for k in range(149):
        n = 40000 if k in (64, 65, 130) else int(rng.integers(1, 300))      # 40,000 x 32 B = 1.22 MiB
        cuts.append((pos, pos + n))
        pos += n
    cuts.append((pos, len(d)))
    assert pos < len(d)
    with _ctx(hicr) as ctx:
        bufs = [torch.from_numpy(w.slot_image(s)).cuda() for s in range(2)]
        ids = [ctx.slot_register(b) for b in bufs]
        for a, b in cuts:
            ctx.memcpy_batch(np.ascontiguousarray(d[a:b]))
        ctx.fence()
        for s in range(2):
            assert bufs[s].cpu().numpy().tobytes() == ref[0][s].tobytes(), "slot %d" % s
        assert [ctx.slot_counters(i) for i in ids] == ref[1][-1]


def test_config1_counters_golden_on_gpu(hicr, golden_dir):
    g = json.load(open(os.path.join(golden_dir, "config1_counters.json")))
    w = W.tiny()
    _, per_epoch, launches = run_gpu(w)
    assert [c[0] for c in per_epoch[-1]] == g["sent"]
    assert [c[1] for c in per_epoch[-1]] == g["recv"]
    assert launches > 0


# ------------------------------------------------------------------- edge cases
def test_zero_size_and_empty_batch(hicr):
    with _ctx(hicr) as ctx:
        a = torch.arange(8, dtype=torch.uint8, device="cuda")
        b = torch.zeros(8, dtype=torch.uint8, device="cuda")
        z = torch.empty(0, dtype=torch.uint8, device="cuda")
        ia, ib, iz = ctx.slot_register(a), ctx.slot_register(b), ctx.slot_register(z)
        ctx.fence()                                         # nothing outstanding: returns at once
        ctx.memcpy_batch(np.zeros(0, dtype=hicr.DESC_DTYPE))  # n == 0 is a no-op
        ctx.fence()
        assert ctx.slot_counters(ia) == (0, 0)
        # zero-size transfers move nothing and still count (reading 4); empty range at the
        # end of a slot and on a zero-size slot are valid
        ctx.memcpy_batch(W.make_descs([ib, ib, iz], [ia, ia, ia], [0, 8, 0], [3, 8, 2], [0, 0, 0]))
        ctx.fence()
        assert b.cpu().tolist() == [0] * 8
        assert ctx.slot_counters(ia) == (3, 0) and ctx.slot_counters(ib) == (0, 2) and ctx.slot_counters(iz) == (0, 1)


def test_rejects_non_device_memory(hicr):
    with _ctx(hicr) as ctx:
        host = np.zeros(64, dtype=np.uint8)
        with pytest.raises(hicr.HicrError) as e:
            ctx.slot_register(int(host.ctypes.data), 64)
        assert e.value.status == hicr.HICR_ERR_UNSUPPORTED_SPACE      # PAPER.md:373 "rejected"


def _error_batch(kind):
    w = W.tiny(n_desc=300, slot_bytes=64 * 1024, max_size=128)
    d = w.epochs[0].copy()
    if kind == "oob_dst":
        d["dst_off"][170] = 64 * 1024 - 3
        d["size"][170] = 4
    elif kind == "oob_src_wrap":
        d["src_off"][170] = 2 ** 64 - 2                               # off + size wraps u64
        d["size"][170] = 8
    elif kind == "bad_slot":
        d["src_slot"][170] = 9
    d["dst_slot"][200] = 77                                           # a later error must not win
    return w, d


@pytest.mark.parametrize("kind,status", [("oob_dst", "HICR_ERR_OUT_OF_BOUNDS"), ("oob_src_wrap", "HICR_ERR_OUT_OF_BOUNDS"),
                                         ("bad_slot", "HICR_ERR_INVALID_SLOT")])
@pytest.mark.parametrize("device_tables", [False, True])
def test_all_or_nothing_errors(hicr, kind, status, device_tables):
    """Reading 10: an invalid descriptor rejects the whole batch, lowest bad index reported;
    the other batches of the epoch are unaffected.  Host tables fail at memcpy_batch,
    device tables at the fence.  Same verdict as the oracle."""
    from oracle import Oracle
    w, bad = _error_batch(kind)
    good = w.epochs[0][:100].copy()
    imgs = [w.slot_image(0), w.slot_image(1)]
    o = Oracle()
    for i in imgs:
        o.slot_register(i)
    orc_status, orc_bad = o.memcpy_batch(bad)
    assert orc_bad == 170
    assert o.memcpy_batch(good)[0] == 0 and o.fence() == 0

    with _ctx(hicr) as ctx:
        bufs = [torch.from_numpy(w.slot_image(s)).cuda() for s in range(2)]
        ids = [ctx.slot_register(b) for b in bufs]
        keep = []
        with pytest.raises(hicr.HicrError) as e:
            if device_tables:
                keep.append(to_device_table(good))
                ctx.memcpy_batch(keep[-1], n=len(good))
                keep.append(to_device_table(bad))
                ctx.memcpy_batch(keep[-1], n=len(bad))
                ctx.fence()
            else:
                ctx.memcpy_batch(good)
                ctx.memcpy_batch(bad)
        assert e.value.status == getattr(hicr, status) == orc_status
        assert e.value.first_bad == 170
        if device_tables:
            assert e.value.batch_index == 1
        else:
            ctx.fence()
        for s in range(2):
            assert bufs[s].cpu().numpy().tobytes() == imgs[s].tobytes()
        assert [ctx.slot_counters(s) for s in ids] == [o.slot_counters(0), o.slot_counters(1)] == [(100, 0), (0, 100)]
        # the context keeps working after a rejected batch
        ctx.memcpy_batch(w.epochs[0][100:200].copy())
        ctx.fence()
        assert ctx.slot_counters(0) == (200, 0)


def test_unregister_then_use_is_invalid_slot(hicr):
    with _ctx(hicr) as ctx:
        a = torch.zeros(64, dtype=torch.uint8, device="cuda")
        b = torch.zeros(64, dtype=torch.uint8, device="cuda")
        ia, ib = ctx.slot_register(a), ctx.slot_register(b)
        ctx.slot_unregister(ia)
        with pytest.raises(hicr.HicrError) as e:
            ctx.slot_unregister(ia)
        assert e.value.status == hicr.HICR_ERR_INVALID_SLOT
        with pytest.raises(hicr.HicrError) as e:
            ctx.memcpy_batch(W.make_descs([ib], [ia], [0], [0], [8]))
        assert e.value.status == hicr.HICR_ERR_INVALID_SLOT
        t = to_device_table(W.make_descs([ib], [ia], [0], [0], [8]))
        ctx.memcpy_batch(t, n=1)
        with pytest.raises(hicr.HicrError) as e:
            ctx.fence()
        assert e.value.status == hicr.HICR_ERR_INVALID_SLOT


def test_register_between_batch_and_fence(hicr):
    """memcpy_batch; slot_register(new); fence: the batch pushed the counters of the slots that
    existed at its launch, the fence must not wait for more, and the new slot reads (0, 0)."""
    w = W.tiny()
    ref = run_oracle(w)
    with _ctx(hicr) as ctx:
        bufs = [torch.from_numpy(w.slot_image(s)).cuda() for s in range(2)]
        ids = [ctx.slot_register(b) for b in bufs]
        t = to_device_table(w.epochs[0])
        ctx.memcpy_batch(t, n=len(w.epochs[0]))
        extra = torch.zeros(128, dtype=torch.uint8, device="cuda")
        ie = ctx.slot_register(extra)
        ctx.fence()
        assert [ctx.slot_counters(i) for i in ids] == ref[1][-1]
        assert ctx.slot_counters(ie) == (0, 0)
        for s in range(2):
            assert bufs[s].cpu().numpy().tobytes() == ref[0][s].tobytes()
        # and hicr_fence_expected after a registration falls back to the full read-back
        ctx.memcpy_batch(t, n=len(w.epochs[0]))
        ie2 = ctx.slot_register(torch.zeros(16, dtype=torch.uint8, device="cuda"))
        ctx.fence_expected(ids[1], 0, 2 * len(w.epochs[0]))
        assert ctx.slot_counters(ids[1]) == (0, 2 * len(w.epochs[0])) and ctx.slot_counters(ie2) == (0, 0)
        ctx.fence()


def test_slot_ids_are_recycled_under_a_new_generation(hicr):
    """Unregistering frees the table index; the next registration takes it under a new id, with
    zeroed counters, and the old id names nothing any more.  A context is not
    capped at HICR_MAX_SLOTS registrations over its lifetime."""
    with _ctx(hicr) as ctx:
        a = torch.arange(64, dtype=torch.uint8, device="cuda")
        b = torch.zeros(64, dtype=torch.uint8, device="cuda")
        ia, ib = ctx.slot_register(a), ctx.slot_register(b)
        assert (ia, ib) == (0, 1)
        ctx.memcpy_batch(W.make_descs([ib], [ia], [0], [0], [8]))
        ctx.fence()
        assert ctx.slot_counters(ib) == (0, 1)
        ctx.slot_unregister(ib)
        c = torch.zeros(64, dtype=torch.uint8, device="cuda")
        ic = ctx.slot_register(c)
        assert ic != ib and ic & 0xfff == ib                       # same index, next generation
        assert ctx.slot_counters(ic) == (0, 0)                      # counters restart at registration
        for table in (False, True):                                 # the old id is dead, on the host and on the device
            d = W.make_descs([ib], [ia], [8], [8], [8])
            with pytest.raises(hicr.HicrError) as e:
                if table:
                    t = to_device_table(d)
                    ctx.memcpy_batch(t, n=1)
                    ctx.fence()
                else:
                    ctx.memcpy_batch(d)
            assert e.value.status == hicr.HICR_ERR_INVALID_SLOT
        with pytest.raises(hicr.HicrError):
            ctx.slot_counters(ib)
        t = to_device_table(W.make_descs([ic, ic], [ia, ia], [0, 16], [32, 0], [16, 5]))
        ctx.memcpy_batch(t, n=2)
        ctx.fence()
        assert ctx.slot_counters(ic) == (0, 2) and ctx.slot_counters(ia) == (3, 0)
        assert c.cpu().tolist()[:21] == list(range(32, 48)) + list(range(5))
        assert b.cpu().tolist()[:8] == list(range(8)) and sum(b.cpu().tolist()[8:]) == 0
        # far more registrations than table rows over the context's lifetime
        last = None
        for k in range(hicr.HICR_MAX_SLOTS + 100):
            last = ctx.slot_register(b)
            ctx.slot_unregister(last)
        assert last >> 12 >= 1000
        ctx.memcpy_batch(W.make_descs([ic], [ia], [40], [0], [4]))
        ctx.fence()
        assert ctx.slot_counters(ic) == (0, 3)


def test_visible_from_another_stream_after_fence(hicr):
    """hicr_fence returns when the last CTA's completion record arrives; the kernel may still be
    running its last instructions.  What the fence promises (hicr.h) must then hold for ANY
    reader: a device-to-host copy and a kernel on OTHER streams, issued right after the fence
    returned, see every byte of the epoch (S5.1 says why).  1,000 rounds of config 1's
    descriptors from four rotating source images (so every round changes the destination bytes),
    the context on a stream of its own."""
    w = W.tiny()
    sa, sb, sc = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    with torch.cuda.stream(sa):
        ctx = hicr.Context(0, sa.cuda_stream)
    try:
        rng = np.random.default_rng(3)
        src_imgs = [rng.integers(0, 256, w.slot_sizes[0], dtype=np.uint8) for _ in range(4)]
        exp = []
        from oracle import Oracle
        for img in src_imgs:
            o = Oracle()
            dst = w.slot_image(1)
            o.slot_register(img.copy())
            o.slot_register(dst)
            assert o.memcpy_batch(w.epochs[0])[0] == 0 and o.fence() == 0
            exp.append(torch.from_numpy(dst.copy()).cuda())
        with torch.cuda.stream(sa):
            srcs = [torch.from_numpy(i).cuda() for i in src_imgs]
            dst0 = torch.from_numpy(w.slot_image(1)).cuda()
            dst = dst0.clone()
            ids = [ctx.slot_register(t) for t in srcs]
            idd = ctx.slot_register(dst)
            tabs = []
            for i in ids:
                d = w.epochs[0].copy()
                d["src_slot"], d["dst_slot"] = i, idd
                tabs.append(to_device_table(d))
        host = torch.empty(dst.numel(), dtype=torch.uint8).pin_memory()
        flag = torch.zeros(1, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        n = len(w.epochs[0])
        for r in range(1000):
            k = r % 4
            ctx.memcpy_batch(tabs[k], n=n)
            ctx.fence()
            # no synchronisation with stream A beyond the fence having returned
            with torch.cuda.stream(sb):
                host.copy_(dst, non_blocking=True)
            with torch.cuda.stream(sc):
                flag += (dst != exp[k]).any().to(torch.int32)
            sb.synchronize()
            assert torch.equal(host, exp[k].cpu()), "round %d: copy on another stream saw stale bytes" % r
        sc.synchronize()
        assert int(flag.item()) == 0, "a kernel on another stream saw stale bytes"
    finally:
        with torch.cuda.stream(sa):
            ctx.close()


def test_tma_min_knob(hicr, monkeypatch):
    """HICR_TMA_MIN, the one tuning knob (read at hicr_init): the large-descriptor cases with
    the bulk-copy path forced on for every aligned chunk and switched off altogether."""
    w = W.heavy_tailed("a", n_slots=6, slot_bytes=16 * W.MiB, src_zone=2 * W.MiB, n_desc=2500, smax=2 * W.MiB, seed=77)
    # make a good share of the large descriptors 16 B-congruent so that the bulk path carries them
    d = w.epochs[0]
    zone = w.meta["src_zone"]
    new = d["src_off"] // 16 * 16 + d["dst_off"] % 16
    new = np.where(new + d["size"] > zone, new - 16, new)
    move = (d["size"] > 8192) & (d["size"] <= zone - 32) & (new >= 0) & (new + d["size"] <= zone)
    d["src_off"][move] = new[move]
    assert int(move.sum()) > 50
    from oracle import hazard
    assert hazard.check(d, w.slot_sizes) is None
    ref = run_oracle(w)
    for v in ("16", "0xffffffff"):
        monkeypatch.setenv("HICR_TMA_MIN", v)
        assert_same(w, ref, run_gpu(w, device_tables=True), "HICR_TMA_MIN=" + v)


# ------------------------------------------------------------ full-size configs
def test_config2_full_size(hicr):
    """BASELINE.json config 2 at full size (2 x 1 GiB, 4 x 65,536 x 4 KiB), in the launch
    configuration bench.py times (device-resident tables, one batch + one fence per set)."""
    w = W.bulk_aligned()
    ref = run_oracle(w)
    got = run_gpu(w, device_tables=True)
    assert_same(w, ref, got)
    assert got[1][-1] == [(4 * 65536, 0), (0, 4 * 65536)]


def test_config4_full_size(hicr):
    """BASELINE.json config 4 at full size: 64 fence epochs x 65,536 descriptors on one
    256 MiB slot; final image and per-epoch counters."""
    w = W.chained_epochs()
    ref = run_oracle(w)
    got = run_gpu(w, device_tables=True)
    assert_same(w, ref, got)
    for k, c in enumerate(got[1]):
        assert c == [(65536 * (k + 1), 65536 * (k + 1))]


@pytest.mark.parametrize("variant", ["a", "b"])
def test_config3_quarter_size(hicr, variant):
    """Config 3's size law and alignment mix at a quarter of the slot count (16 x 256 MiB =
    4 GiB, 25,000 descriptors, sizes up to 16 MiB), whole-image parity."""
    w = W.heavy_tailed(variant, n_slots=16, n_desc=25000)
    ref = run_oracle(w)
    got = run_gpu(w, device_tables=True)
    assert_same(w, ref, got)


# ------------------------------------------------------------ host tables on several host threads
def test_large_host_table_parity_and_late_error(hicr):
    """A host table long enough for the threaded check-and-stage path (hicr_stage.cu: pieces of
    4096 descriptors claimed by the caller and the helper threads): same image and counters
    as the oracle; with two bad descriptors in late pieces the LOWEST index is reported,
    nothing is copied or counted, and the context keeps working."""
    from oracle import Oracle
    w = W.bulk_aligned(n_desc=50000, slot_bytes=256 * W.MiB, page=1024, n_sets=1)
    ref = run_oracle(w)
    got = run_gpu(w, device_tables=False)
    assert_same(w, ref, got, "threaded host table")

    bad = w.epochs[0].copy()
    bad["src_off"][45000] = 2 ** 63                                   # a later piece
    bad["dst_slot"][30001] = 5                                        # the lowest bad index
    o = Oracle()
    for s in range(2):
        o.slot_register(w.slot_image(s))
    orc_status, orc_bad = o.memcpy_batch(bad)
    assert orc_bad == 30001
    with _ctx(hicr) as ctx:
        bufs = [torch.from_numpy(w.slot_image(s)).cuda() for s in range(2)]
        ids = [ctx.slot_register(b) for b in bufs]
        with pytest.raises(hicr.HicrError) as e:
            ctx.memcpy_batch(bad)
        assert e.value.status == hicr.HICR_ERR_INVALID_SLOT == orc_status
        assert e.value.first_bad == 30001
        ctx.fence()
        for s in range(2):
            assert bufs[s].cpu().numpy().tobytes() == w.slot_image(s).tobytes()
        assert [ctx.slot_counters(s) for s in ids] == [(0, 0), (0, 0)]
        ctx.memcpy_batch(w.epochs[0])
        ctx.fence()
        assert [ctx.slot_counters(s) for s in ids] == [(50000, 0), (0, 50000)]
        for s in range(2):
            assert bufs[s].cpu().numpy().tobytes() == ref[0][s].tobytes()


def test_chain_host_tables_static_hand_out(hicr):
    """Config 4's shape through HOST tables: the host counts the batch as team-sized, so the
    kernel runs without barrier and with the static hand-out; 6 chained epochs."""
    w = W.chained_epochs(n_epochs=6, n_desc=20000, slot_bytes=32 * W.MiB)
    assert_same(w, run_oracle(w), run_gpu(w, device_tables=False), "chain, host tables")


@pytest.mark.timeout(1800)
@pytest.mark.parametrize("variant", ["a", "b"])
def test_config3_full_size(hicr, variant):
    """BASELINE.json config 3 (variants 3a and 3b, reading 19) at FULL size -- 64 slots x 256 MiB,
    100,000 descriptors (3a) / every log-uniform draw that fits (3b), one device-resident batch, one
    fence: the launch configuration bench.py times.
    The oracle gets the same descriptors one destination slot at a time, against slots trimmed
    to the zones they touch (the destination slot whole, every slot's 32 MiB source zone), so
    16 GiB never has to sit in host memory twice; every byte of every slot is compared."""
    from oracle import Oracle
    w = W.heavy_tailed(variant)
    d = w.epochs[0]
    zone = w.meta["src_zone"]
    n_slots = len(w.slot_sizes)
    assert int((d["src_off"] + d["size"]).max()) <= zone and int(d["dst_off"].min()) >= zone
    with _ctx(hicr) as ctx:
        bufs = []
        for s in range(n_slots):
            bufs.append(torch.from_numpy(w.slot_image(s)).cuda())
        ids = [ctx.slot_register(b) for b in bufs]
        t = to_device_table(d)
        ctx.memcpy_batch(t, n=len(d))
        ctx.fence()
        got_cnt = [ctx.slot_counters(s) for s in ids]
        assert ctx.launch_count() == 1
        sources = [w.slot_image(s)[:zone].copy() for s in range(n_slots)]
        for s in range(n_slots):
            sel = d[d["dst_slot"] == s].copy()
            o = Oracle()
            img = w.slot_image(s)
            assert o.slot_register(img) == 0
            for z in sources:
                o.slot_register(z)
            sel["dst_slot"] = 0
            sel["src_slot"] = sel["src_slot"] + 1
            assert o.memcpy_batch(np.ascontiguousarray(sel))[0] == 0 and o.fence() == 0
            assert o.slot_counters(0)[1] == len(sel) == got_cnt[s][1]
            assert bufs[s].cpu().numpy().tobytes() == img.tobytes(), "slot %d differs from the oracle" % s
            o.close()
        sent = np.bincount(d["src_slot"], minlength=n_slots)
        assert [c[0] for c in got_cnt] == sent.tolist()


# ------------------------------------------------------------ stream-ordered and expected-count fences
def test_fence_async_chain(hicr):
    """hicr_fence_async: config 4's dependency chain with stream-ordered
    fences between the epochs and one blocking fence at the end leaves the image and the
    counters the oracle reaches with a blocking fence per epoch."""
    w = W.chained_epochs(n_epochs=8, n_desc=20000, slot_bytes=32 * W.MiB)
    ref_imgs, ref_cnt = run_oracle(w)
    with _ctx(hicr) as ctx:
        buf = torch.from_numpy(w.slot_image(0)).cuda()
        sid = ctx.slot_register(buf)
        keep = []
        for e in w.epochs:
            keep.append(to_device_table(e))
            ctx.memcpy_batch(keep[-1], n=len(e))
            ctx.fence_async()
        ctx.fence()
        assert buf.cpu().numpy().tobytes() == ref_imgs[0].tobytes()
        assert ctx.slot_counters(sid) == ref_cnt[-1][0] == (8 * 20000, 8 * 20000)


def test_chain_recorded_once_replayed_twice(hicr):
    """hicr_graph_* (config 4 "as one CUDA graph"): the chain of epochs recorded
    once and enqueued with one call leaves image and counters as the oracle's epoch-by-epoch run;
    a second launch replays the same epochs on the image the first one left (the oracle does the
    same); a replay with a bad descriptor reports it at the fence with its batch index and leaves
    that batch without effect; recording refuses what it cannot replay."""
    w = W.chained_epochs(n_epochs=8, n_desc=20000, slot_bytes=32 * W.MiB)
    imgs = [w.slot_image(0)]
    o = Oracle()
    o.slot_register(imgs[0])
    with _ctx(hicr) as c0:
        with pytest.raises(hicr.HicrError) as e:
            c0.graph_begin(16)                                                 # the legacy default stream
        assert e.value.status == hicr.HICR_ERR_INVALID_ARG
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream), hicr.Context(0, stream.cuda_stream) as ctx:
        buf = torch.from_numpy(w.slot_image(0)).cuda()
        sid = ctx.slot_register(buf)
        keep = [to_device_table(e) for e in w.epochs]
        stream.synchronize()
        ctx.graph_begin(20000)
        for t, e in zip(keep, w.epochs):
            ctx.memcpy_batch(t, n=len(e))
            ctx.fence_async()
        with pytest.raises(hicr.HicrError) as e:
            ctx.memcpy_batch(np.ascontiguousarray(w.epochs[0]))               # a host table cannot be replayed
        assert e.value.status == hicr.HICR_ERR_INVALID_ARG
        with pytest.raises(hicr.HicrError) as e:
            ctx.fence()                                                        # nor can a blocking fence be recorded
        assert e.value.status == hicr.HICR_ERR_BUSY
        g = ctx.graph_end()
        l0 = ctx.launch_count()
        for rep in (1, 2):
            for ep in w.epochs:
                assert o.memcpy_batch(np.ascontiguousarray(ep))[0] == oracle.OK and o.fence() == oracle.OK
            g.launch()
            ctx.fence()
            assert buf.cpu().numpy().tobytes() == imgs[0].tobytes(), "launch %d" % rep
            assert ctx.slot_counters(sid) == o.slot_counters(0) == (rep * 8 * 20000, rep * 8 * 20000)
        assert ctx.launch_count() - l0 == 16
        # a bad descriptor in epoch 5 of the recorded tables: found by the replay, reported at the fence
        bad = np.ascontiguousarray(w.epochs[5]).copy()
        bad["size"][777] = 1 << 40
        keep[5].copy_(to_device_table(bad))
        for k, ep in enumerate(w.epochs):
            rc, idx = o.memcpy_batch(bad if k == 5 else np.ascontiguousarray(ep))
            assert (rc, idx) == ((oracle.ERR_OUT_OF_BOUNDS, 777) if k == 5 else (oracle.OK, None))
            assert o.fence() == oracle.OK
        g.launch()
        with pytest.raises(hicr.HicrError) as e:
            ctx.fence()
        assert (e.value.status, e.value.batch_index, e.value.first_bad) == (hicr.HICR_ERR_OUT_OF_BOUNDS, 5, 777)
        assert buf.cpu().numpy().tobytes() == imgs[0].tobytes()
        assert ctx.slot_counters(sid) == o.slot_counters(0)
        # a changed slot table makes the recording stale
        extra = torch.zeros(16, dtype=torch.uint8, device="cuda")
        ctx.slot_register(extra)
        with pytest.raises(hicr.HicrError) as e:
            g.launch()
        assert e.value.status == hicr.HICR_ERR_INVALID_ARG
        g.close()


def test_fence_expected(hicr):
    """hicr_fence_expected ("until the expected number of incoming and outgoing data
    transfers have been completed"): returns once the slot's cumulative counts are reached,
    reports INVALID_ARG when the enqueued work can never reach them, and leaves the epoch
    to an ordinary fence.  Reading of DESIGN.md S2 (unpinned by the paper)."""
    w = W.tiny(n_desc=600, slot_bytes=256 * 1024, max_size=300)
    parts = np.array_split(w.epochs[0], 3)
    ref = run_oracle(w)
    with _ctx(hicr) as ctx:
        bufs = [torch.from_numpy(w.slot_image(s)).cuda() for s in range(2)]
        ids = [ctx.slot_register(b) for b in bufs]
        assert ctx.fence_expected(ids[1], 0, 0) is None                       # already true, nothing outstanding
        with pytest.raises(hicr.HicrError) as e:
            ctx.fence_expected(ids[1], 0, 1)                                  # nothing outstanding: never
        assert e.value.status == hicr.HICR_ERR_INVALID_ARG
        keep = [to_device_table(p) for p in parts]
        for t, p in zip(keep, parts):
            ctx.memcpy_batch(t, n=len(p))
        ctx.fence_expected(ids[1], 0, len(parts[0]))                          # at least the first batch is in
        assert ctx.slot_counters(ids[1])[1] >= len(parts[0])
        ctx.fence_expected(ids[1], 0, 600)
        ctx.fence_expected(ids[0], 600, 0)
        assert ctx.slot_counters(ids[1]) == (0, 600) and ctx.slot_counters(ids[0]) == (600, 0)
        for s in range(2):
            assert bufs[s].cpu().numpy().tobytes() == ref[0][s].tobytes()
        with pytest.raises(hicr.HicrError) as e:
            ctx.fence_expected(ids[1], 0, 601)                                # everything is complete: never
        assert e.value.status == hicr.HICR_ERR_INVALID_ARG
        ctx.fence()
        # a rejected device batch counts nothing: the expected fence returns its deferred error
        bad = parts[0].copy()
        bad["src_slot"][5] = 99
        t = to_device_table(bad)
        ctx.memcpy_batch(t, n=len(bad))
        with pytest.raises(hicr.HicrError) as e:
            ctx.fence_expected(ids[1], 0, 600 + len(bad))
        assert e.value.status == hicr.HICR_ERR_INVALID_SLOT and e.value.first_bad == 5
        assert ctx.slot_counters(ids[1]) == (0, 600)


@pytest.mark.timeout(600)
def test_no_access_past_the_end_of_a_slot():
    """Slots that end on the last mapped byte before unmapped virtual addresses: a kernel that
    reads or writes one 16-byte granule too far faults.  Runs in a subprocess (a fault poisons
    the CUDA context); see tests/guard_page_check.py."""
    import subprocess
    import sys
    r = subprocess.run([sys.executable, os.path.join(os.path.dirname(__file__), "guard_page_check.py")],
                       capture_output=True, text=True, timeout=550)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "guard page check ok" in r.stdout


@pytest.mark.timeout(900)
def test_randomized_mixes(hicr):
    """60 seeded workloads drawn from all four generators with random sizes of slot, batch and
    descriptor (team, warp and chunk classes mixed, 1 to 3 batches per epoch), each through
    host tables and device tables: every byte and counter equals the oracle's."""
    rng = np.random.default_rng(W.BASE_SEED + 99)
    done = 0
    while done < 60:
        seed, kind = int(rng.integers(1, 1 << 30)), int(rng.integers(0, 4))
        try:
            if kind == 0:
                w = W.heavy_tailed("a", n_slots=int(rng.integers(2, 70)), slot_bytes=int(rng.integers(3, 9)) * W.MiB,
                                   src_zone=W.MiB, n_desc=int(rng.integers(1, 6000)),
                                   smax=int(rng.choice([300, 9000, 200000, 900000])), seed=seed)
            elif kind == 1:
                w = W.tiny(n_desc=int(rng.integers(1, 3000)), slot_bytes=int(rng.integers(1, 5)) * W.MiB,
                           max_size=int(rng.choice([16, 256, 300, 4096, 20000])), seed=seed)
            elif kind == 2:
                w = W.chained_epochs(n_epochs=int(rng.integers(2, 6)), n_desc=int(rng.integers(10, 30000)),
                                     slot_bytes=16 * W.MiB, smin=int(rng.choice([1, 8])),
                                     smax=int(rng.choice([16, 256, 1000])), seed=seed)
            else:
                w = W.bulk_aligned(n_desc=int(rng.integers(1, 5000)), slot_bytes=64 * W.MiB,
                                   page=int(rng.choice([16, 256, 1024, 4096, 16384])), n_sets=2, seed=seed)
        except ValueError:
            continue                                   # the draw does not fit its slots
        ref = run_oracle(w)
        for dev in (False, True):
            got = run_gpu(w, device_tables=dev, split=int(rng.integers(1, 4)))
            assert_same(w, ref, got, "kind %d seed %d device_tables %s" % (kind, seed, dev))
        done += 1


def test_chain_refused_after_the_chunk_queue_moved(hicr):
    """A recorded chain names the chunk queue it was recorded with.  An ordinary batch larger than
    anything before re-allocates that queue; the chain must then be refused, not replayed into
    freed memory."""
    MiB = W.MiB
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream), hicr.Context(0, stream.cuda_stream) as ctx:
        a = torch.zeros(8 * MiB, dtype=torch.uint8, device="cuda")
        b = torch.from_numpy(W.random_bytes(W.rng_for(9, 1), 8 * MiB)).cuda()
        sa, sb = ctx.slot_register(a), ctx.slot_register(b)
        large = W.make_descs([sa] * 4, [sb] * 4, [k * MiB + 3 for k in range(4)], [k * MiB + 5 for k in range(4)], [MiB - 64] * 4)
        t = to_device_table(large)
        stream.synchronize()
        ctx.graph_begin(16)
        ctx.memcpy_batch(t, n=4)
        g = ctx.graph_end()
        g.launch()
        ctx.fence()
        for k in range(4):
            assert torch.equal(a[k * MiB + 3: (k + 1) * MiB - 61], b[k * MiB + 5: (k + 1) * MiB - 59])
        # 20,000 descriptors: far more than the 16 the recording sized the queue for
        many = W.make_descs([sa] * 20000, [sb] * 20000, np.arange(20000) * 64 + 4 * MiB, np.arange(20000) * 64, [48] * 20000)
        t2 = to_device_table(many)
        ctx.memcpy_batch(t2, n=20000)
        ctx.fence()
        with pytest.raises(hicr.HicrError) as e:
            g.launch()
        assert e.value.status == hicr.HICR_ERR_INVALID_ARG
        ctx.fence()
        g.close()
        # a chain recorded now replays
        ctx.graph_begin(16)
        ctx.memcpy_batch(t, n=4)
        g2 = ctx.graph_end()
        a.zero_()
        g2.launch()
        ctx.fence()
        assert torch.equal(a[3: MiB - 61], b[5: MiB - 59])
        g2.close()


def test_recording_refuses_channel_and_global_calls(hicr):
    """While a chain is being recorded every other call that would put work on the stream
    returns HICR_ERR_BUSY (hicr.h): channels, MPSC sets and the global-slot calls too."""
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream), hicr.Context(0, stream.cuda_stream) as ctx:
        ring, src, dst = (torch.zeros(4096, dtype=torch.uint8, device="cuda") for _ in range(3))
        r, s, d = (ctx.slot_register(x) for x in (ring, src, dst))
        ch = ctx.channel_create(r, 64, 16)
        r2 = ctx.slot_register(torch.zeros(4096, dtype=torch.uint8, device="cuda"))
        m = ctx.mpsc_create([r2], 64, 16)
        handle = ctx.global_volunteer(1, 0, s)
        one = to_device_table(W.make_descs([d], [s], [1024], [0], [16]))
        stream.synchronize()
        ctx.graph_begin(16)
        ctx.memcpy_batch(one, n=1)
        refused = [
            lambda: ch.push(s, 0, 4), lambda: ch.pop(d, 0, 4), lambda: ch.stream(s, 0, d, 0, [4, 4]),
            lambda: ch.locking_stream([s], d, 0, 8, 4), lambda: m.stream([s], [d], 8, 4),
            lambda: ctx.channel_create(r2, 64, 16), lambda: ctx.mpsc_create([r2], 64, 16),
            lambda: ctx.global_fence_begin(), lambda: ctx.global_fence_end(np.zeros(1, dtype=hicr.GLOBAL_COUNT_DTYPE)),
            lambda: ctx.global_counters(s), lambda: ctx.global_exchange(1, [handle]),
        ]
        for k, call in enumerate(refused):
            with pytest.raises(hicr.HicrError) as e:
                call()
            assert e.value.status == hicr.HICR_ERR_BUSY, k
        g = ctx.graph_end()
        g.close()
        # and the same calls work once the recording is over
        src.copy_(torch.arange(4096, dtype=torch.int32, device="cuda").to(torch.uint8))
        assert ch.push(s, 0, 4) == 4 and ch.pop(d, 0, 4) == 4
        assert torch.equal(dst[:256], src[:256])
        m.close()
        ch.close()
