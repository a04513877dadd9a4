"""hicr_memcpy_batch_noalloc against the context path (hicr_memcpy_batch + hicr_fence).

Who needs the entry point under test: a program that cannot let this library allocate -- all of
its HBM sits in a pool of its own, so a cudaMalloc from inside the library fails, or it runs
a loop next to other streams and cannot take the device-wide stall of the cudaMalloc / cudaFree
with which hicr_memcpy_batch grows its chunk queue.  The entry point keeps that queue (and
its counters and control words) in an array compiled into the library, so it must behave the
same on every call although the array still holds the call before: that is what two calls in a
row, with different batches, check here.  Both paths are this library's CUDA code; the context
path is itself compared with the CPU definition elsewhere in tests/.

Bit-exact, as everywhere in this suite: every byte of every slot, every counter, the status and
the index of the first bad descriptor.  The file sorts last on purpose (pytest -x would hide
everything after a failure here) and does not depend on having run after, or before, any other test.
"""
import numpy as np
import pytest

import workloads as W
from parity import to_device_table

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

MiB = 1 << 20


@pytest.fixture(scope="module")
def hicr():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import paper_2509_01425_b200 as h
    return h


def _batch(seed, n_desc, n_slots, slot_bytes, src_zone):
    """Mixed batch: power-law sizes 16 B .. 1 MiB at byte-granular offsets (team-, warp- and
    chunk-sized descriptors, ragged tails), plus a few zero-size descriptors."""
    w = W.heavy_tailed("a", n_slots=n_slots, slot_bytes=slot_bytes, src_zone=src_zone, n_desc=n_desc, smin=16,
                       smax=MiB, seed=seed)
    d = w.epochs[0]
    z = W.make_descs([1, 2, 0], [0, 2, 1], [slot_bytes, 5, 0], [0, slot_bytes, 7], [0, 0, 0])
    return w, np.concatenate([d[: n_desc // 2], z, d[n_desc // 2:]])


class _NoAlloc:
    """The caller's side of the entry point: its own slot array, counters and result words."""

    def __init__(self, hicr, bufs):
        self.hicr = hicr
        rows = np.zeros(len(bufs), dtype=hicr.RAW_SLOT_DTYPE)
        rows["base"] = [b.data_ptr() for b in bufs]
        rows["size"] = [b.numel() for b in bufs]
        self.n_slots = len(bufs)
        self.d_slots = torch.from_numpy(rows.view(np.uint8).copy()).cuda()
        self.d_counters = torch.zeros(2 * len(bufs), dtype=torch.int64, device="cuda")
        self.d_result = torch.full((2,), -99, dtype=torch.int64, device="cuda")

    def run(self, descs):
        t = to_device_table(descs) if len(descs) else torch.empty(0, dtype=torch.uint8, device="cuda")
        self.d_result.fill_(-99)
        self.hicr.memcpy_batch_noalloc(0, torch.cuda.current_stream().cuda_stream, self.d_slots.data_ptr(), self.n_slots,
                                       t.data_ptr(), len(descs), self.d_counters.data_ptr(), self.d_result.data_ptr())
        torch.cuda.synchronize()
        res = self.d_result.cpu().tolist()
        cnt = self.d_counters.cpu().tolist()
        return res, [(cnt[2 * s], cnt[2 * s + 1]) for s in range(self.n_slots)]


def _context_path(hicr, ctx, ids, descs):
    """Existing path: device-resident table, error (if any) at the fence."""
    t = to_device_table(descs)
    res = [hicr.HICR_OK, 0]
    try:
        ctx.memcpy_batch(t, n=len(descs))
        ctx.fence()
    except hicr.HicrError as e:
        res = [e.status, e.first_bad]
    return res, [ctx.slot_counters(s) for s in ids]


def _same_images(a_bufs, b_bufs, what):
    for s, (a, b) in enumerate(zip(a_bufs, b_bufs)):
        a, b = a.cpu().numpy(), b.cpu().numpy()
        if a.tobytes() != b.tobytes():
            diff = np.nonzero(a != b)[0]
            raise AssertionError("%s: slot %d differs at %d bytes, first at %d" % (what, s, diff.size, diff[0]))


def test_two_calls_in_a_row_match_the_context_path(hicr):
    n_slots, slot_bytes, src_zone = 6, 24 * MiB, 2 * MiB
    w, first = _batch(101, 3000, n_slots, slot_bytes, src_zone)
    _, second = _batch(202, 700, n_slots, slot_bytes, src_zone)
    assert (first["size"] > 128 * 1024).sum() > (second["size"] > 128 * 1024).sum() > 0   # the second queue is shorter
    bad = second.copy()
    bad["size"][400] = slot_bytes                       # out of bounds at 400 ...
    bad["dst_slot"][450] = n_slots                      # ... and an unknown slot later: 400 is reported
    imgs = [w.slot_image(s) for s in range(n_slots)]
    ref_bufs = [torch.from_numpy(i).cuda() for i in imgs]
    got_bufs = [torch.from_numpy(i).cuda() for i in imgs]
    na = _NoAlloc(hicr, got_bufs)
    with hicr.Context(0, torch.cuda.current_stream().cuda_stream) as ctx:
        ids = [ctx.slot_register(b) for b in ref_bufs]
        assert ids == list(range(n_slots))
        for what, descs in (("first call", first), ("second call", second), ("rejected call", bad),
                            ("call after a rejected one", first[::-1].copy()), ("empty call", first[:0])):
            ref = _context_path(hicr, ctx, ids, descs) if len(descs) else ([hicr.HICR_OK, 0], [ctx.slot_counters(s) for s in ids])
            got = na.run(descs)
            assert got == ref, what
            _same_images(ref_bufs, got_bufs, what)
        assert ref[1][0][0] > 0 and got[0] == [hicr.HICR_OK, 0]
    assert na.run(bad)[0] == [hicr.HICR_ERR_OUT_OF_BOUNDS, 400]


def test_sizes_beyond_the_fixed_scratch_are_refused(hicr):
    bufs = [torch.zeros(64 * MiB + 4096, dtype=torch.uint8, device="cuda"), torch.ones(64 * MiB + 4096, dtype=torch.uint8, device="cuda")]
    na = _NoAlloc(hicr, bufs)
    one = W.make_descs([0], [1], [0], [0], [16])
    stream = torch.cuda.current_stream().cuda_stream
    t = to_device_table(one)
    for n_slots, n in ((2, hicr.HICR_NOALLOC_MAX_DESCS + 1), (hicr.HICR_NOALLOC_MAX_SLOTS + 1, 1)):
        with pytest.raises(hicr.HicrError) as e:
            hicr.memcpy_batch_noalloc(0, stream, na.d_slots.data_ptr(), n_slots, t.data_ptr(), n, na.d_counters.data_ptr(),
                                      na.d_result.data_ptr())
        assert e.value.status == hicr.HICR_ERR_NO_CAPACITY
    # more chunks than the queue holds: known on the device only, reported like a bad descriptor
    n_big = hicr.HICR_NOALLOC_MAX_CHUNKS // 512 + 1                 # 65 descriptors of 64 MiB = 512 chunks each
    big = W.make_descs([0] * n_big, [1] * n_big, [0] * n_big, [0] * n_big, [64 * MiB] * n_big)   # (never copied: overlap is moot)
    res, cnt = na.run(big)
    assert res[0] == hicr.HICR_ERR_NO_CAPACITY and 0 <= res[1] < n_big
    assert cnt == [(0, 0), (0, 0)] and int(bufs[0].max()) == 0
    # and the call after it works
    res, cnt = na.run(W.make_descs([0], [1], [3], [0], [100001]))
    assert res == [hicr.HICR_OK, 0] and cnt == [(0, 1), (1, 0)]
    assert int(bufs[0].sum()) == 100001
