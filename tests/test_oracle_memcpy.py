"""Pins for the CPU oracle's memcpy / fence (CPU only, -m "not gpu").

The oracle is pinned against things other than itself: values printed by the paper /
SPEC (tests/golden/), the closed form evaluated by numpy slicing, libc memmove,
exhaustive brute force over every (dst_off, src_off, size) on tiny slots, order
independence, the paper's broadcast listing and closed-form counter values.
"""
import ctypes
import itertools
import json
import os

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import Oracle, hazard


def _bytes(s):
    return np.frombuffer(s.encode("ascii"), dtype=np.uint8).copy()


STATUS = {"ok": oracle.OK, "out_of_bounds": oracle.ERR_OUT_OF_BOUNDS, "invalid_slot": oracle.ERR_INVALID_SLOT}


def _one(dst, dst_off, src, src_off, size):
    return W.make_descs([dst], [src], [dst_off], [src_off], [size])


# ------------------------------------------------------------------ printed examples
def test_golden_memcpy_examples(golden_dir):
    cases = json.load(open(os.path.join(golden_dir, "memcpy_examples.json")))["cases"]
    assert len(cases) >= 8
    for c in cases:
        o = Oracle()
        arrs = [_bytes(s) for s in c["slots"]]
        ids = [o.slot_register(a) for a in arrs]
        m = c["memcpy"]
        rc, bad = o.memcpy_batch(_one(ids[m["dst"]], m["dst_off"], ids[m["src"]], m["src_off"], m["size"]))
        assert rc == STATUS[c["status"]], c["cite"]
        if rc != oracle.OK:
            assert bad == 0
        assert o.fence() == oracle.OK
        for a, e in zip(arrs, c["expect"]):
            assert a.tobytes().decode("ascii") == e, c["cite"]


def test_golden_broadcast(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "broadcast.json")))
    msg = _bytes(g["message"])
    o = Oracle()
    m = o.slot_register(msg)
    rng = np.random.default_rng(7)
    dsts = [rng.integers(0, 256, g["destination_size"], dtype=np.uint8) for _ in range(g["n_destinations"])]
    before = [d.copy() for d in dsts]
    ids = [o.slot_register(d) for d in dsts]
    # the paper issues one memcpy per destination and a single fence after the loops
    for i in ids:
        rc, _ = o.memcpy_batch(_one(i, 0, m, 0, msg.size))
        assert rc == oracle.OK
    assert o.pending() == len(ids)
    assert o.fence() == oracle.OK
    for d, b in zip(dsts, before):
        assert d[: msg.size].tobytes() == msg.tobytes()
        assert d[msg.size:].tobytes() == b[msg.size:].tobytes()
    assert o.slot_counters(m) == (len(ids), 0)
    for i in ids:
        assert o.slot_counters(i) == (0, 1)


# ------------------------------------------------------------ exhaustive brute force
def _libc_memmove(dst_arr, dst_off, src_arr, src_off, n):
    ctypes.memmove(dst_arr.ctypes.data + dst_off, src_arr.ctypes.data + src_off, n)


@pytest.mark.parametrize("L", [17, 21])
def test_exhaustive_two_slots(L):
    """Every (dst_off, src_off, size) on two L-byte slots: valid ones equal the closed form
    out[x] = src0[src_off + x - dst_off] on the destination range, dst0[x] elsewhere (and
    libc memmove); invalid ones are rejected with nothing changed."""
    rng = np.random.default_rng(L)
    src0 = rng.integers(0, 256, L, dtype=np.uint8)
    dst0 = rng.integers(0, 256, L, dtype=np.uint8)
    n_ok = n_bad = 0
    for do, so, n in itertools.product(range(L + 2), range(L + 2), range(L + 2)):
        s, d = src0.copy(), dst0.copy()
        o = Oracle()
        si, di = o.slot_register(s), o.slot_register(d)
        rc, bad = o.memcpy_batch(_one(di, do, si, so, n))
        valid = do + n <= L and so + n <= L
        if valid:
            assert rc == oracle.OK
            exp = dst0.copy()
            exp[do: do + n] = src0[so: so + n]
            mm = dst0.copy()
            _libc_memmove(mm, do, src0, so, n)
            assert d.tobytes() == exp.tobytes() == mm.tobytes()
            assert s.tobytes() == src0.tobytes()
            n_ok += 1
        else:
            assert rc == oracle.ERR_OUT_OF_BOUNDS and bad == 0
            assert d.tobytes() == dst0.tobytes() and s.tobytes() == src0.tobytes()
            assert o.pending() == 0
            n_bad += 1
        o.close()
    assert n_ok > 1000 and n_bad > 1000


def test_exhaustive_one_slot_memmove():
    """Same slot as source and destination: every (dst_off, src_off, size), overlapping or
    not, equals libc memmove ('as if through an intermediate buffer')."""
    L = 16
    base = np.arange(L, dtype=np.uint8) * 7 + 3
    for do, so, n in itertools.product(range(L + 1), range(L + 1), range(L + 1)):
        if do + n > L or so + n > L:
            continue
        a = base.copy()
        o = Oracle()
        i = o.slot_register(a)
        rc, _ = o.memcpy_batch(_one(i, do, i, so, n))
        assert rc == oracle.OK
        mm = base.copy()
        _libc_memmove(mm, do, mm, so, n)
        assert a.tobytes() == mm.tobytes()
        o.close()


# ---------------------------------------------------------------- bounds and errors
def test_bounds_do_not_wrap_u64():
    a = np.zeros(8, dtype=np.uint8)
    b = np.ones(8, dtype=np.uint8)
    o = Oracle()
    ia, ib = o.slot_register(a), o.slot_register(b)
    big = (1 << 64) - 1
    for d in (_one(ib, big, ia, 0, 2), _one(ib, 0, ia, big, 2), _one(ib, 0, ia, 0, big), _one(ib, 4, ia, 0, big - 2)):
        rc, bad = o.memcpy_batch(d)
        assert rc == oracle.ERR_OUT_OF_BOUNDS and bad == 0
    assert b.tolist() == [1] * 8


def test_invalid_slot_and_unregister():
    a = np.zeros(8, dtype=np.uint8)
    b = np.ones(8, dtype=np.uint8)
    o = Oracle()
    ia, ib = o.slot_register(a), o.slot_register(b)
    assert o.memcpy_batch(_one(ib, 0, 99, 0, 1))[0] == oracle.ERR_INVALID_SLOT
    assert o.memcpy_batch(_one(99, 0, ia, 0, 1))[0] == oracle.ERR_INVALID_SLOT
    assert o.slot_unregister(ia) == oracle.OK
    assert o.slot_unregister(ia) == oracle.ERR_INVALID_SLOT  # double unregister
    assert o.memcpy_batch(_one(ib, 0, ia, 0, 1))[0] == oracle.ERR_INVALID_SLOT
    assert b.tolist() == [1] * 8


def test_batch_is_all_or_nothing_and_reports_first_bad():
    """Reading 10: one invalid descriptor rejects the whole batch, nothing is copied,
    nothing is counted; first_bad is the lowest bad index and the status is that one's."""
    w = W.tiny(n_desc=64, slot_bytes=64 * 1024, max_size=512)
    d = w.epochs[0].copy()
    d["src_slot"][40] = 77          # invalid slot at 40
    d["dst_off"][23] = 64 * 1024    # out of bounds at 23 (size >= 1)
    imgs = [w.slot_image(0), w.slot_image(1)]
    before = [i.copy() for i in imgs]
    o = Oracle()
    for i in imgs:
        o.slot_register(i)
    rc, bad = o.memcpy_batch(d)
    assert (rc, bad) == (oracle.ERR_OUT_OF_BOUNDS, 23)
    assert o.pending() == 0 and o.fence() == oracle.OK
    assert all(a.tobytes() == b.tobytes() for a, b in zip(imgs, before))
    assert o.slot_counters(0) == (0, 0) and o.slot_counters(1) == (0, 0)
    d["dst_off"][23] = 0
    d["size"][23] = 0
    rc, bad = o.memcpy_batch(d)
    assert (rc, bad) == (oracle.ERR_INVALID_SLOT, 40)


# ------------------------------------------------- batches: invariants and closed forms
def _run(w, epochs=None, perm_seed=None):
    imgs = [w.slot_image(s) for s in range(len(w.slot_sizes))]
    o = Oracle()
    for i in imgs:
        o.slot_register(i)
    for e in (w.epochs if epochs is None else epochs):
        if perm_seed is not None:
            e = e[np.random.default_rng(perm_seed).permutation(len(e))]
        rc, _ = o.memcpy_batch(np.ascontiguousarray(e))
        assert rc == oracle.OK
        assert o.fence() == oracle.OK
    return o, imgs


def _numpy_epoch(imgs0, descs):
    """Independent statement of one epoch under the precondition: every destination range
    takes the source bytes of the image at the START of the epoch (numpy slicing)."""
    out = [i.copy() for i in imgs0]
    for d in descs:
        n = int(d["size"])
        out[d["dst_slot"]][int(d["dst_off"]): int(d["dst_off"]) + n] = \
            imgs0[d["src_slot"]][int(d["src_off"]): int(d["src_off"]) + n]
    return out


SMALL = {
    "tiny": lambda: W.tiny(),
    "bulk": lambda: W.bulk_aligned(n_desc=256, slot_bytes=4 * W.MiB, n_sets=1),
    "heavy_a": lambda: W.heavy_tailed("a", n_slots=6, slot_bytes=2 * W.MiB, src_zone=256 * W.KiB,
                                      n_desc=1500, smax=128 * W.KiB),
    "heavy_b": lambda: W.heavy_tailed("b", n_slots=6, slot_bytes=2 * W.MiB, src_zone=256 * W.KiB,
                                      n_desc=1500, smax=128 * W.KiB),
}


@pytest.mark.parametrize("name", sorted(SMALL))
def test_epoch_equals_closed_form_and_invariants(name):
    w = SMALL[name]()
    d = w.epochs[0]
    assert hazard.check(d, w.slot_sizes) is None
    imgs0 = [w.slot_image(s) for s in range(len(w.slot_sizes))]
    o, imgs = _run(w, epochs=[d])
    exp = _numpy_epoch(imgs0, d)
    for a, e in zip(imgs, exp):
        assert a.tobytes() == e.tobytes()
    # north_star invariants, stated with a mask: destination bytes equal source bytes,
    # bytes outside every destination range are unchanged
    for s in range(len(imgs)):
        touched = np.zeros(w.slot_sizes[s], dtype=bool)
        for x in d[d["dst_slot"] == s]:
            touched[int(x["dst_off"]): int(x["dst_off"] + x["size"])] = True
        assert np.array_equal(imgs[s][~touched], imgs0[s][~touched])
    for x in d[:: max(1, len(d) // 200)]:
        n = int(x["size"])
        assert np.array_equal(imgs[x["dst_slot"]][int(x["dst_off"]): int(x["dst_off"]) + n],
                              imgs0[x["src_slot"]][int(x["src_off"]): int(x["src_off"]) + n])
    # counters: closed form = descriptor counts per source slot / per destination slot
    ns = len(imgs)
    sent = np.bincount(d["src_slot"], minlength=ns)
    recv = np.bincount(d["dst_slot"], minlength=ns)
    got = [o.slot_counters(s) for s in range(ns)]
    assert [g[0] for g in got] == sent.tolist() and [g[1] for g in got] == recv.tolist()
    assert sum(g[0] for g in got) == sum(g[1] for g in got) == len(d)


@pytest.mark.parametrize("name", ["tiny", "heavy_a"])
def test_order_independence(name):
    """Under the epoch precondition the image does not depend on the order in which the
    descriptors are applied (completion order is not guaranteed)."""
    w = SMALL[name]()
    _, ref = _run(w)
    for seed in (1, 2, 3):
        _, got = _run(w, perm_seed=seed)
        for a, b in zip(ref, got):
            assert a.tobytes() == b.tobytes()


def test_config1_counters_golden(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "config1_counters.json")))
    w = W.tiny()
    assert w.n_descs == g["n_desc"]
    o, _ = _run(w)
    assert [o.slot_counters(s)[0] for s in (0, 1)] == g["sent"]
    assert [o.slot_counters(s)[1] for s in (0, 1)] == g["recv"]


def test_zero_size_counts_but_moves_nothing():
    """Reading 4: a zero-size memcpy is a no-op that still counts."""
    a = np.arange(8, dtype=np.uint8)
    b = np.zeros(8, dtype=np.uint8)
    o = Oracle()
    ia, ib = o.slot_register(a), o.slot_register(b)
    rc, _ = o.memcpy_batch(W.make_descs([ib, ib], [ia, ia], [0, 8], [3, 8], [0, 0]))
    assert rc == oracle.OK and o.fence() == oracle.OK
    assert b.tolist() == [0] * 8
    assert o.slot_counters(ia) == (2, 0) and o.slot_counters(ib) == (0, 2)


def test_counters_change_only_at_fence_and_empty_fence_is_noop():
    w = W.tiny(n_desc=32, slot_bytes=16 * 1024, max_size=256)
    imgs = [w.slot_image(0), w.slot_image(1)]
    o = Oracle()
    for i in imgs:
        o.slot_register(i)
    assert o.fence() == oracle.OK                      # nothing outstanding
    assert o.slot_counters(0) == (0, 0)
    assert o.memcpy_batch(w.epochs[0])[0] == oracle.OK
    assert o.slot_counters(0) == (0, 0) and o.pending() == 32
    assert o.fence() == oracle.OK
    assert o.slot_counters(0) == (32, 0) and o.slot_counters(1) == (0, 32) and o.pending() == 0
    snap = [i.copy() for i in imgs]
    assert o.fence() == oracle.OK
    assert o.slot_counters(0) == (32, 0) and o.slot_counters(1) == (0, 32)
    assert all(a.tobytes() == b.tobytes() for a, b in zip(imgs, snap))


def test_chained_epochs_against_numpy_and_per_epoch_counters():
    """Config 4 scaled down: a missed or early-visible byte in epoch k corrupts every
    later epoch, so the final image checks ordering across fences.  Reading 8: after
    fence k (0-based) sent = recv = n_desc * (k + 1) on the single slot."""
    w = W.chained_epochs(n_epochs=6, n_desc=512, slot_bytes=256 * W.KiB)
    img = w.slot_image(0)
    cur = [img.copy()]
    o = Oracle()
    o.slot_register(img)
    for k, e in enumerate(w.epochs):
        assert hazard.check(e, w.slot_sizes) is None
        assert o.memcpy_batch(e)[0] == oracle.OK and o.fence() == oracle.OK
        assert o.slot_counters(0) == (512 * (k + 1), 512 * (k + 1))
        cur = _numpy_epoch(cur, e)
    assert img.tobytes() == cur[0].tobytes()
    # the chain is real: every epoch-(k+1) source range lies inside one epoch-k destination
    for k in range(1, len(w.epochs)):
        p, c = w.epochs[k - 1], w.epochs[k]
        order = np.argsort(p["dst_off"])
        lo, hi = p["dst_off"][order], (p["dst_off"] + p["size"])[order]
        j = np.searchsorted(lo, c["src_off"], side="right") - 1
        assert np.all(j >= 0) and np.all(c["src_off"] + c["size"] <= hi[j])


def test_parallel_memcpy_baseline_equals_the_oracle():
    """oracle/parallel_memcpy.c (bench.py's cpu_baseline_parallel: libc memcpy per descriptor on
    all host cores) is a timing baseline, not the oracle; its image must still
    be the oracle's on inputs that meet the epoch precondition, for 1 and for several threads."""
    import workloads as W
    for w in (W.heavy_tailed("a", n_slots=6, slot_bytes=4 * W.MiB, src_zone=W.MiB, n_desc=2000, smax=300000),
              W.chained_epochs(n_epochs=1, n_desc=5000, slot_bytes=4 * W.MiB)):
        ref = [w.slot_image(s) for s in range(len(w.slot_sizes))]
        o = Oracle()
        for a in ref:
            o.slot_register(a)
        assert o.memcpy_batch(w.epochs[0])[0] == oracle.OK
        for threads in (1, 5):
            got = [w.slot_image(s) for s in range(len(w.slot_sizes))]
            oracle.parallel_memcpy_batch(got, w.epochs[0], threads)
            assert all(a.tobytes() == b.tobytes() for a, b in zip(ref, got))
