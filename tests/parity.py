"""Parity harness: run one seeded workload through the CPU oracle and through the CUDA
library (via the C-ABI binding) and compare byte for byte.  Test infrastructure only.

The two sides share nothing but the input arrays drawn by ``workloads``.
"""
from __future__ import annotations

import numpy as np

import oracle
import workloads as W
from oracle import Oracle


def run_oracle(w: W.CopyWorkload, epochs=None):
    """Returns (final images, [counters after each fence]); counters = list of (sent, recv)."""
    imgs = [w.slot_image(s) for s in range(len(w.slot_sizes))]
    o = Oracle()
    for i in imgs:
        o.slot_register(i)
    per_epoch = []
    for e in (w.epochs if epochs is None else epochs):
        rc, bad = o.memcpy_batch(np.ascontiguousarray(e))
        assert rc == oracle.OK, (rc, bad)
        assert o.fence() == oracle.OK
        per_epoch.append([o.slot_counters(s) for s in range(len(imgs))])
    return imgs, per_epoch


def to_device_table(descs: np.ndarray):
    import torch
    return torch.from_numpy(np.ascontiguousarray(descs).view(np.uint8).copy()).cuda()


def run_gpu(w: W.CopyWorkload, epochs=None, device_tables=False, split=1):
    """Same workload through hicr_slot_register / hicr_memcpy_batch / hicr_fence.
    ``split`` > 1 submits each epoch as that many batches before its single fence."""
    import torch
    import paper_2509_01425_b200 as hicr

    ctx = hicr.Context(0, torch.cuda.current_stream().cuda_stream)
    try:
        bufs = [torch.from_numpy(w.slot_image(s)).cuda() for s in range(len(w.slot_sizes))]
        ids = [ctx.slot_register(b) for b in bufs]
        assert ids == list(range(len(bufs)))
        per_epoch = []
        keep = []
        for e in (w.epochs if epochs is None else epochs):
            parts = np.array_split(np.ascontiguousarray(e), split) if split > 1 else [np.ascontiguousarray(e)]
            for part in parts:
                part = np.ascontiguousarray(part)
                if device_tables:
                    t = to_device_table(part)
                    keep.append(t)
                    ctx.memcpy_batch(t, n=len(part))
                else:
                    ctx.memcpy_batch(part)
            ctx.fence()
            keep.clear()
            per_epoch.append([ctx.slot_counters(s) for s in ids])
        torch.cuda.synchronize()
        imgs = [b.cpu().numpy() for b in bufs]
        launches = ctx.launch_count()
    finally:
        ctx.close()
    return imgs, per_epoch, launches


def assert_same(w, ref, got, what=""):
    ref_imgs, ref_cnt = ref
    got_imgs, got_cnt = got[0], got[1]
    assert len(ref_imgs) == len(got_imgs)
    for s, (a, b) in enumerate(zip(ref_imgs, got_imgs)):
        if a.tobytes() != b.tobytes():
            diff = np.nonzero(a != b)[0]
            raise AssertionError("%s %s: slot %d differs at %d bytes, first at %d (oracle %d, cuda %d)"
                                 % (w.name, what, s, diff.size, diff[0], a[diff[0]], b[diff[0]]))
    assert ref_cnt == got_cnt, "%s %s: counters differ" % (w.name, what)
