"""ctypes binding of include/hicr.h: argument marshalling only.

Every step of the path (validation, binning, copies, counters, fence, channel push/pop)
runs in the CUDA library; nothing here touches slot bytes.  PyTorch is used by callers
for device memory and streams; this module only takes ``tensor.data_ptr()``.

There is no CPU fallback: if libhicr_b200.so cannot be loaded (or built with nvcc) the
import of this module raises, and without a CUDA device ``Context()`` raises
``HicrError(HICR_ERR_CUDA)``.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

# status codes (include/hicr.h)
HICR_OK = 0
HICR_ERR_INVALID_ARG = -1
HICR_ERR_INVALID_SLOT = -2
HICR_ERR_OUT_OF_BOUNDS = -3
HICR_ERR_UNSUPPORTED_SPACE = -4
HICR_ERR_NO_CAPACITY = -5
HICR_ERR_CUDA = -6
HICR_ERR_BUSY = -7
HICR_ERR_ILLEGAL_DIRECTION = -8
HICR_ERR_DUPLICATE_KEY = -9
HICR_ERR_TIMEOUT = -10
HICR_MAX_SLOTS = 4096
HICR_GLOBAL_HANDLE_BYTES = 256

# hicr_global_count_t: one line of a global fence's count exchange
GLOBAL_COUNT_DTYPE = np.dtype([("tag", "<u8"), ("key", "<u8"), ("sent", "<u8"), ("recv", "<u8")])
assert GLOBAL_COUNT_DTYPE.itemsize == 32

# hicr_desc_t: dst_slot, src_slot, dst_off, src_off, size (PAPER.md:532 argument order)
DESC_DTYPE = np.dtype(
    [("dst_slot", "<u4"), ("src_slot", "<u4"), ("dst_off", "<u8"), ("src_off", "<u8"), ("size", "<u8")]
)
assert DESC_DTYPE.itemsize == 32

EXPORTS = (
    "hicr_init", "hicr_finalize", "hicr_strerror", "hicr_last_cuda_error",
    "hicr_slot_register", "hicr_slot_unregister", "hicr_slot_counters",
    "hicr_memcpy_batch", "hicr_fence", "hicr_fence_error", "hicr_fence_async", "hicr_fence_expected",
    "hicr_memcpy_batch_noalloc",
    "hicr_channel_create", "hicr_channel_destroy", "hicr_channel_counters",
    "hicr_channel_push", "hicr_channel_pop", "hicr_channel_stream",
    "hicr_mpsc_create", "hicr_mpsc_destroy", "hicr_mpsc_counters", "hicr_mpsc_stream",
    "hicr_mpsc_locking_stream",
    "hicr_instance_set", "hicr_global_volunteer", "hicr_global_exchange", "hicr_global_lookup",
    "hicr_global_fence_begin", "hicr_global_fence_end", "hicr_global_counters",
    "hicr_graph_begin", "hicr_graph_end", "hicr_graph_launch", "hicr_graph_destroy",
    "hicr_launch_count", "hicr_profile_enable", "hicr_profile_read",
)


def _load() -> ctypes.CDLL:
    path = _build.LIB
    if _build.is_stale():
        # sources newer than the library (or no library): rebuild with nvcc, loudly
        path = _build.build()
    lib = ctypes.CDLL(path)
    vp, u32, u64, i32 = ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int
    P = ctypes.POINTER
    sig = {
        "hicr_init": (i32, [P(vp), i32, vp]),
        "hicr_finalize": (i32, [vp]),
        "hicr_strerror": (ctypes.c_char_p, [i32]),
        "hicr_last_cuda_error": (ctypes.c_char_p, [vp]),
        "hicr_slot_register": (i32, [vp, vp, u64, P(u32)]),
        "hicr_slot_unregister": (i32, [vp, u32]),
        "hicr_slot_counters": (i32, [vp, u32, P(u64), P(u64)]),
        "hicr_memcpy_batch": (i32, [vp, vp, u64, i32, P(u64)]),
        "hicr_memcpy_batch_noalloc": (i32, [i32, vp, vp, u32, vp, u64, vp, vp]),
        "hicr_fence": (i32, [vp]),
        "hicr_fence_error": (i32, [vp, P(u64), P(u64)]),
        "hicr_fence_async": (i32, [vp]),
        "hicr_fence_expected": (i32, [vp, u32, u64, u64]),
        "hicr_channel_create": (i32, [vp, u32, u64, u64, P(vp)]),
        "hicr_channel_destroy": (i32, [vp]),
        "hicr_channel_counters": (i32, [vp, P(u64), P(u64)]),
        "hicr_channel_push": (i32, [vp, u32, u64, u64, P(u64)]),
        "hicr_channel_pop": (i32, [vp, u32, u64, u64, P(u64)]),
        "hicr_channel_stream": (i32, [vp, u32, u64, u32, u64, vp, u64]),
        "hicr_mpsc_create": (i32, [vp, u32, vp, u64, u64, P(vp)]),
        "hicr_mpsc_destroy": (i32, [vp]),
        "hicr_mpsc_counters": (i32, [vp, u32, P(u64), P(u64)]),
        "hicr_mpsc_stream": (i32, [vp, vp, vp, vp, vp, u64, u64]),
        "hicr_mpsc_locking_stream": (i32, [vp, u32, vp, u32, u64, u64, u64]),
        "hicr_instance_set": (i32, [vp, u32, u32]),
        "hicr_global_volunteer": (i32, [vp, u64, u64, u32, vp]),
        "hicr_global_exchange": (i32, [vp, u64, vp, u64, vp]),
        "hicr_global_lookup": (i32, [vp, u64, u64, P(u32)]),
        "hicr_global_fence_begin": (i32, [vp, vp, u64, P(u64)]),
        "hicr_global_fence_end": (i32, [vp, vp, u64, u32]),
        "hicr_global_counters": (i32, [vp, u32, P(u64), P(u64)]),
        "hicr_graph_begin": (i32, [vp, u64]),
        "hicr_graph_end": (i32, [vp, P(vp)]),
        "hicr_graph_launch": (i32, [vp]),
        "hicr_graph_destroy": (i32, [vp]),
        "hicr_launch_count": (i32, [vp, P(u64)]),
        "hicr_profile_enable": (i32, [vp, i32]),
        "hicr_profile_read": (i32, [vp, P(ctypes.c_float)]),
    }
    for name in EXPORTS:
        fn = getattr(lib, name)  # AttributeError = a declared symbol is missing: fail loudly
        fn.restype, fn.argtypes = sig[name]
    return lib


lib = _load()
LIB_PATH = _build.LIB
# the calls of a step, through the CPython C API instead of ctypes (csrc/hicr_pyext.c); the
# extension links against the library loaded above
from . import _hicr_step as _step  # noqa: E402


class HicrError(RuntimeError):
    def __init__(self, status: int, where: str, first_bad=None, batch_index=None, detail: str = ""):
        self.status = status
        self.first_bad = first_bad
        self.batch_index = batch_index
        msg = "%s: %s (%d)" % (where, lib.hicr_strerror(status).decode(), status)
        if first_bad is not None:
            msg += " first_bad=%d" % first_bad
        if detail:
            msg += " [" + detail + "]"
        super().__init__(msg)


# hicr_raw_slot_t: one row of the slot array hicr_memcpy_batch_noalloc takes
RAW_SLOT_DTYPE = np.dtype([("base", "<u8"), ("size", "<u8")])
HICR_NOALLOC_MAX_DESCS = 65536
HICR_NOALLOC_MAX_SLOTS = 1024
HICR_NOALLOC_MAX_CHUNKS = 32768


def memcpy_batch_noalloc(device: int, stream: int, d_slots: int, n_slots: int, d_descs: int, n: int,
                         d_counters: int, d_result: int) -> None:
    """hicr_memcpy_batch_noalloc: the batch for callers that may not allocate (a process whose
    HBM belongs to its own pool, a loop that cannot take cudaMalloc's device-wide stall).  All
    pointers are device addresses as ints (``tensor.data_ptr()``); ``stream`` a cudaStream_t as
    int.  Enqueues and returns; status and first bad index arrive in ``d_result``.  Raises
    HicrError for what the host can refuse (limits, NULL, CUDA errors)."""
    rc = lib.hicr_memcpy_batch_noalloc(device, stream, d_slots, n_slots, d_descs, n, d_counters, d_result)
    if rc != HICR_OK:
        raise HicrError(rc, "hicr_memcpy_batch_noalloc")


def _slot_ids(ids) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(ids, dtype=np.uint32))


class Context:
    """hicr_init / hicr_finalize.  ``stream``: a cudaStream_t handle as int (e.g.
    ``torch.cuda.current_stream().cuda_stream``); 0 = the legacy default stream."""

    def __init__(self, device: int = 0, stream: int = 0):
        h = ctypes.c_void_p()
        rc = lib.hicr_init(ctypes.byref(h), device, ctypes.c_void_p(stream))
        if rc != HICR_OK:
            raise HicrError(rc, "hicr_init")
        self._h = h
        self._hv = h.value   # the handle as a plain int, for the C-API entry points
        self._keep = {}      # slot id -> object that owns the storage (kept alive)
        self._children = []

    # ---- plumbing
    def close(self):
        if getattr(self, "_h", None):
            for c in list(self._children):
                c.close()
            lib.hicr_finalize(self._h)
            self._h = None
            self._keep.clear()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _fail(self, rc, where, **kw):
        detail = lib.hicr_last_cuda_error(self._h).decode() if rc == HICR_ERR_CUDA else ""
        raise HicrError(rc, where, detail=detail, **kw)

    # ---- slots
    def slot_register(self, buf, size=None) -> int:
        """hicr_slot_register.  ``buf``: a torch tensor (its storage bytes from
        data_ptr(), numel*element_size bytes, must be contiguous) or an int device
        address with ``size``."""
        if isinstance(buf, int):
            ptr, nbytes, owner = buf, int(size), None
        else:
            if not buf.is_contiguous():
                raise ValueError("slot storage must be contiguous")
            nbytes = buf.numel() * buf.element_size() if size is None else int(size)
            ptr, owner = (buf.data_ptr() if nbytes else 0), buf
        out = ctypes.c_uint32()
        rc = lib.hicr_slot_register(self._h, ctypes.c_void_p(ptr), nbytes, ctypes.byref(out))
        if rc != HICR_OK:
            self._fail(rc, "hicr_slot_register")
        self._keep[out.value] = owner
        return out.value

    def slot_unregister(self, slot: int):
        rc = lib.hicr_slot_unregister(self._h, slot)
        if rc != HICR_OK:
            self._fail(rc, "hicr_slot_unregister")
        self._keep.pop(slot, None)

    def slot_counters(self, slot: int):
        s, r = ctypes.c_uint64(), ctypes.c_uint64()
        rc = lib.hicr_slot_counters(self._h, slot, ctypes.byref(s), ctypes.byref(r))
        if rc != HICR_OK:
            self._fail(rc, "hicr_slot_counters")
        return s.value, r.value

    # ---- memcpy + fence
    def memcpy_batch(self, descs, n=None):
        """hicr_memcpy_batch.  ``descs``: numpy array of DESC_DTYPE (host table), or a
        torch CUDA tensor / int device address of ``n`` 32-byte descriptors (device
        table; must stay alive until the fence)."""
        if type(descs) is int:                  # device address: nothing to marshal
            ptr, cnt, dev = descs, n, 1
        elif isinstance(descs, np.ndarray):
            if descs.dtype != DESC_DTYPE or not descs.flags.c_contiguous:
                raise ValueError("host descriptor table must be a contiguous DESC_DTYPE array")
            cnt = descs.size if n is None else int(n)
            ptr, dev = (descs.ctypes.data if cnt else 0), 0
        else:
            nbytes = descs.numel() * descs.element_size()
            cnt = nbytes // 32 if n is None else int(n)
            ptr, dev = (descs.data_ptr() if cnt else 0), 1
        r = _step.memcpy_batch(self._hv, ptr, cnt, dev)
        if r:
            self._fail(r[0], "hicr_memcpy_batch", first_bad=r[1])

    def fence(self):
        rc = _step.fence(self._hv)
        if rc:
            b, i = ctypes.c_uint64(), ctypes.c_uint64()
            lib.hicr_fence_error(self._h, ctypes.byref(b), ctypes.byref(i))
            self._fail(rc, "hicr_fence", first_bad=i.value, batch_index=b.value)

    def fence_async(self):
        rc = _step.fence_async(self._hv)
        if rc:
            self._fail(rc, "hicr_fence_async")

    def fence_expected(self, slot: int, sent: int, recv: int):
        rc = lib.hicr_fence_expected(self._h, slot, sent, recv)
        if rc != HICR_OK:
            b, i = ctypes.c_uint64(), ctypes.c_uint64()
            lib.hicr_fence_error(self._h, ctypes.byref(b), ctypes.byref(i))
            self._fail(rc, "hicr_fence_expected", first_bad=i.value, batch_index=b.value)

    # ---- replayable chains (hicr_graph_*)
    def graph_begin(self, max_descs_per_batch: int):
        rc = lib.hicr_graph_begin(self._h, max_descs_per_batch)
        if rc != HICR_OK:
            self._fail(rc, "hicr_graph_begin")

    def graph_end(self) -> "Graph":
        h = ctypes.c_void_p()
        rc = lib.hicr_graph_end(self._h, ctypes.byref(h))
        if rc != HICR_OK:
            self._fail(rc, "hicr_graph_end")
        g = Graph(self, h)
        self._children.append(g)
        return g

    # ---- Global Memory Slots (the local halves; collective.py carries the bytes between instances)
    def instance_set(self, instance: int, n_instances: int):
        rc = lib.hicr_instance_set(self._h, instance, n_instances)
        if rc != HICR_OK:
            self._fail(rc, "hicr_instance_set")

    def global_volunteer(self, tag: int, key: int, local_slot: int) -> bytes:
        """hicr_global_volunteer: the 256-byte handle of ``local_slot`` as (tag, key)."""
        buf = ctypes.create_string_buffer(HICR_GLOBAL_HANDLE_BYTES)
        rc = lib.hicr_global_volunteer(self._h, tag, key, local_slot, buf)
        if rc != HICR_OK:
            self._fail(rc, "hicr_global_volunteer")
        return buf.raw

    def global_exchange(self, tag: int, handles) -> list:
        """hicr_global_exchange: ``handles`` = the handles of all instances in the agreed order;
        returns this context's Global Memory Slot id of each."""
        handles = list(handles)
        n = len(handles)
        if any(len(h) != HICR_GLOBAL_HANDLE_BYTES for h in handles):
            raise ValueError("a global handle is %d bytes" % HICR_GLOBAL_HANDLE_BYTES)
        blob = ctypes.create_string_buffer(b"".join(handles), max(1, n * HICR_GLOBAL_HANDLE_BYTES))
        out = (ctypes.c_uint32 * max(1, n))()
        rc = lib.hicr_global_exchange(self._h, tag, blob, n, out)
        if rc != HICR_OK:
            self._fail(rc, "hicr_global_exchange")
        ids = [int(out[i]) for i in range(n)]
        for g in ids:
            self._keep[g] = None
        return ids

    def global_lookup(self, tag: int, key: int) -> int:
        out = ctypes.c_uint32()
        rc = lib.hicr_global_lookup(self._h, tag, key, ctypes.byref(out))
        if rc != HICR_OK:
            self._fail(rc, "hicr_global_lookup")
        return out.value

    def global_fence_begin(self, defer_error: bool = False):
        """hicr_global_fence_begin: the blocking local fence, then this context's lines of the
        count exchange (GLOBAL_COUNT_DTYPE).  A deferred error of the epoch is raised here, or --
        ``defer_error`` -- returned as the second element of (lines, HicrError or None), so that a
        collective caller can finish the exchange with its peers before raising it."""
        cap = 64
        while True:
            out = np.zeros(cap, dtype=GLOBAL_COUNT_DTYPE)
            n = ctypes.c_uint64()
            rc = lib.hicr_global_fence_begin(self._h, ctypes.c_void_p(out.ctypes.data), cap, ctypes.byref(n))
            if rc == HICR_ERR_NO_CAPACITY and n.value > cap:
                cap = int(n.value)
                continue
            err = None
            if rc != HICR_OK:
                b, i = ctypes.c_uint64(), ctypes.c_uint64()
                lib.hicr_fence_error(self._h, ctypes.byref(b), ctypes.byref(i))
                detail = lib.hicr_last_cuda_error(self._h).decode() if rc == HICR_ERR_CUDA else ""
                err = HicrError(rc, "hicr_global_fence_begin", first_bad=i.value, batch_index=b.value, detail=detail)
                if not defer_error or rc == HICR_ERR_CUDA:
                    raise err
            lines = out[: n.value].copy()
            return (lines, err) if defer_error else lines

    def global_fence_end(self, all_counts: np.ndarray, timeout_ms: int = 0):
        a = np.ascontiguousarray(all_counts, dtype=GLOBAL_COUNT_DTYPE)
        rc = lib.hicr_global_fence_end(self._h, ctypes.c_void_p(a.ctypes.data if a.size else 0), a.size, timeout_ms)
        if rc != HICR_OK:
            self._fail(rc, "hicr_global_fence_end")

    def global_counters(self, slot: int):
        s, r = ctypes.c_uint64(), ctypes.c_uint64()
        rc = lib.hicr_global_counters(self._h, slot, ctypes.byref(s), ctypes.byref(r))
        if rc != HICR_OK:
            self._fail(rc, "hicr_global_counters")
        return s.value, r.value

    # ---- channels
    def channel_create(self, ring: int, token_bytes: int, capacity: int) -> "Channel":
        h = ctypes.c_void_p()
        rc = lib.hicr_channel_create(self._h, ring, token_bytes, capacity, ctypes.byref(h))
        if rc != HICR_OK:
            self._fail(rc, "hicr_channel_create")
        ch = Channel(self, h)
        self._children.append(ch)
        return ch

    def mpsc_create(self, rings, token_bytes: int, capacity: int) -> "Mpsc":
        ids = _slot_ids(rings)
        h = ctypes.c_void_p()
        rc = lib.hicr_mpsc_create(self._h, ids.size, ctypes.c_void_p(ids.ctypes.data), token_bytes, capacity,
                                  ctypes.byref(h))
        if rc != HICR_OK:
            self._fail(rc, "hicr_mpsc_create")
        m = Mpsc(self, h, ids.size)
        self._children.append(m)
        return m

    # ---- measurement hooks
    def launch_count(self) -> int:
        v = ctypes.c_uint64()
        rc = lib.hicr_launch_count(self._h, ctypes.byref(v))
        if rc != HICR_OK:
            self._fail(rc, "hicr_launch_count")
        return v.value

    def profile_enable(self, on: bool = True):
        rc = lib.hicr_profile_enable(self._h, 1 if on else 0)
        if rc != HICR_OK:
            self._fail(rc, "hicr_profile_enable")

    def profile_read(self):
        ms = (ctypes.c_float * 4)()
        rc = lib.hicr_profile_read(self._h, ms)
        if rc != HICR_OK:
            self._fail(rc, "hicr_profile_read")
        return [float(x) for x in ms]


class Graph:
    """A recorded chain of batches (hicr_graph_*)."""

    def __init__(self, ctx: Context, h):
        self._ctx, self._h = ctx, h

    def launch(self):
        rc = lib.hicr_graph_launch(self._h)
        if rc != HICR_OK:
            self._ctx._fail(rc, "hicr_graph_launch")

    def close(self):
        if self._h:
            lib.hicr_graph_destroy(self._h)
            self._h = None
            if self in self._ctx._children:
                self._ctx._children.remove(self)


class Channel:
    """SPSC channel handle (hicr_channel_*)."""

    def __init__(self, ctx: Context, h):
        self._ctx, self._h, self._hv = ctx, h, h.value

    def close(self):
        if self._h:
            lib.hicr_channel_destroy(self._h)
            self._h = self._hv = None
            if self in self._ctx._children:
                self._ctx._children.remove(self)

    def counters(self):
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        rc = lib.hicr_channel_counters(self._h, ctypes.byref(a), ctypes.byref(b))
        if rc != HICR_OK:
            self._ctx._fail(rc, "hicr_channel_counters")
        return a.value, b.value

    def push(self, src: int, src_off: int, n_tokens: int) -> int:
        k = _step.channel_push(self._hv, src, src_off, n_tokens)
        if k < 0:
            self._ctx._fail(k, "hicr_channel_push")
        return k

    def pop(self, dst: int, dst_off: int, max_tokens: int) -> int:
        k = _step.channel_pop(self._hv, dst, dst_off, max_tokens)
        if k < 0:
            self._ctx._fail(k, "hicr_channel_pop")
        return k

    def locking_stream(self, src_slots, dst: int, dst_off: int, tokens_per_producer: int, max_batch: int):
        """hicr_mpsc_locking_stream: len(src_slots) producers share this channel's ring."""
        ids = _slot_ids(src_slots)
        rc = lib.hicr_mpsc_locking_stream(self._h, ids.size, ctypes.c_void_p(ids.ctypes.data), dst, dst_off,
                                          tokens_per_producer, max_batch)
        if rc != HICR_OK:
            self._ctx._fail(rc, "hicr_mpsc_locking_stream")

    def stream(self, src: int, src_off: int, dst: int, dst_off: int, batch_tokens):
        b = np.ascontiguousarray(np.asarray(batch_tokens, dtype=np.uint64))
        rc = lib.hicr_channel_stream(self._h, src, src_off, dst, dst_off,
                                     ctypes.c_void_p(b.ctypes.data if b.size else 0), b.size)
        if rc != HICR_OK:
            self._ctx._fail(rc, "hicr_channel_stream")


class Mpsc:
    """Non-locking MPSC handle (hicr_mpsc_*)."""

    def __init__(self, ctx: Context, h, producers: int):
        self._ctx, self._h, self.producers = ctx, h, producers

    def close(self):
        if self._h:
            lib.hicr_mpsc_destroy(self._h)
            self._h = None
            if self in self._ctx._children:
                self._ctx._children.remove(self)

    def counters(self, producer: int):
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        rc = lib.hicr_mpsc_counters(self._h, producer, ctypes.byref(a), ctypes.byref(b))
        if rc != HICR_OK:
            self._ctx._fail(rc, "hicr_mpsc_counters")
        return a.value, b.value

    def stream(self, src_slots, dst_slots, tokens_per_producer: int, max_batch: int, src_offs=None, dst_offs=None):
        s, d = _slot_ids(src_slots), _slot_ids(dst_slots)
        if s.size != self.producers or d.size != self.producers:
            raise ValueError("need one source and one sink slot per producer")
        offs = []
        for o in (src_offs, dst_offs):
            a = None if o is None else np.ascontiguousarray(np.asarray(o, dtype=np.uint64))
            if a is not None and a.size != self.producers:
                raise ValueError("need one offset per producer")
            offs.append(a)
        so, do = (ctypes.c_void_p(a.ctypes.data) if a is not None else None for a in offs)
        rc = lib.hicr_mpsc_stream(self._h, ctypes.c_void_p(s.ctypes.data), so, ctypes.c_void_p(d.ctypes.data), do,
                                  tokens_per_producer, max_batch)
        if rc != HICR_OK:
            self._ctx._fail(rc, "hicr_mpsc_stream")
