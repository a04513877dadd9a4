"""CPU oracle for the HiCR memory-slot memcpy / fence / channel path (TEST INFRASTRUCTURE).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_2509_01425_b200``) never does, and this package never imports the product.

``hicr_oracle.c`` holds the arithmetic (plain single-threaded byte loops, each function
citing the PAPER.md passage it follows); this module only compiles it with gcc and
marshals numpy arrays into it.  ``hazard.py`` is the epoch-precondition checker of
SURVEY.md S8(c) point 5.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hicr_oracle.c")
_LIB = os.path.join(_HERE, "libhicr_oracle.so")

# status codes as hicr_oracle.c defines them
OK = 0
ERR_INVALID_ARG = -1
ERR_INVALID_SLOT = -2
ERR_OUT_OF_BOUNDS = -3
ERR_NO_CAPACITY = -5
ERR_ILLEGAL_DIRECTION = -8   # "Global-to-Global operations are not permitted"
ERR_DUPLICATE_KEY = -9       # a (tag, key) pair names one global slot; used by world.py

# descriptor layout = the paper's argument order dst, dst_off, src, src_off, size
DESC_DTYPE = np.dtype(
    [("dst_slot", "<u4"), ("src_slot", "<u4"), ("dst_off", "<u8"), ("src_off", "<u8"), ("size", "<u8")]
)
assert DESC_DTYPE.itemsize == 32

_PM_SRC = os.path.join(_HERE, "parallel_memcpy.c")
_PM_LIB = os.path.join(_HERE, "libparallel_memcpy.so")

_lock = threading.Lock()
_lib = None
_pm_lib = None


def build(force: bool = False) -> str:
    """Compile hicr_oracle.c into libhicr_oracle.so with gcc (building is not using)."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + ".tmp.%d" % os.getpid()
            subprocess.check_call(
                ["gcc", "-O2", "-std=c99", "-Wall", "-Wextra", "-shared", "-fPIC", "-o", tmp, _SRC]
            )
            os.replace(tmp, _LIB)
        if force or not os.path.exists(_PM_LIB) or os.path.getmtime(_PM_LIB) < os.path.getmtime(_PM_SRC):
            tmp = _PM_LIB + ".tmp.%d" % os.getpid()
            subprocess.check_call(
                ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-shared", "-fPIC", "-pthread", "-o", tmp, _PM_SRC]
            )
            os.replace(tmp, _PM_LIB)
    return _LIB


def parallel_memcpy_batch(images, descs: np.ndarray, threads: int) -> None:
    """The stronger CPU baseline of SURVEY.md S8(d) (parallel_memcpy.c): libc memcpy per
    descriptor over ``threads`` host threads.  Timing baseline only -- no validation, no
    counters; ``descs`` must be a set the oracle accepts and that meets the epoch precondition."""
    global _pm_lib
    if _pm_lib is None:
        build()
        _pm_lib = ctypes.CDLL(_PM_LIB)
        _pm_lib.parallel_memcpy_batch.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int]
    assert descs.dtype == DESC_DTYPE and descs.flags.c_contiguous
    bases = (ctypes.c_void_p * len(images))(*[a.ctypes.data if a.size else 0 for a in images])
    rc = _pm_lib.parallel_memcpy_batch(bases, descs.ctypes.data, descs.size, int(threads))
    if rc != 0:
        raise RuntimeError("parallel_memcpy_batch: could not start its threads")


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    u8p = ctypes.c_void_p
    u32, u64 = ctypes.c_uint32, ctypes.c_uint64
    P = ctypes.POINTER
    lib.oracle_new.restype = ctypes.c_void_p
    lib.oracle_new.argtypes = []
    lib.oracle_free.restype = None
    lib.oracle_free.argtypes = [ctypes.c_void_p]
    lib.oracle_slot_register.argtypes = [ctypes.c_void_p, u8p, u64, P(u32)]
    lib.oracle_slot_register_global.argtypes = [ctypes.c_void_p, ctypes.c_void_p, u32, P(u32)]
    lib.oracle_slot_is_global.argtypes = [ctypes.c_void_p, u32]
    lib.oracle_slot_global_counters.argtypes = [ctypes.c_void_p, u32, P(u64), P(u64)]
    lib.oracle_slot_unregister.argtypes = [ctypes.c_void_p, u32]
    lib.oracle_slot_counters.argtypes = [ctypes.c_void_p, u32, P(u64), P(u64)]
    lib.oracle_memcpy_batch.argtypes = [ctypes.c_void_p, ctypes.c_void_p, u64, P(u64)]
    lib.oracle_fence.argtypes = [ctypes.c_void_p]
    lib.oracle_pending.restype = u64
    lib.oracle_pending.argtypes = [ctypes.c_void_p]
    lib.oracle_channel_create.argtypes = [ctypes.c_void_p, u32, u64, u64, P(u32)]
    lib.oracle_channel_counters.argtypes = [ctypes.c_void_p, u32, P(u64), P(u64)]
    lib.oracle_channel_push.argtypes = [ctypes.c_void_p, u32, u32, u64, u64, P(u64)]
    lib.oracle_channel_pop.argtypes = [ctypes.c_void_p, u32, u32, u64, u64, P(u64)]
    _lib = lib
    return lib


class Oracle:
    """One oracle context: slots over caller-owned numpy uint8 arrays, batches, fence, channels."""

    def __init__(self):
        self._lib = _load()
        self._ctx = self._lib.oracle_new()
        self._keep = []  # registered arrays stay alive as long as the context

    def close(self):
        if self._ctx:
            self._lib.oracle_free(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- slots ---------------------------------------------------------------------
    def slot_register(self, arr: np.ndarray) -> int:
        assert arr.dtype == np.uint8 and arr.ndim == 1 and arr.flags.c_contiguous and arr.flags.writeable
        out = ctypes.c_uint32()
        ptr = arr.ctypes.data if arr.size else 0
        rc = self._lib.oracle_slot_register(self._ctx, ptr, arr.size, ctypes.byref(out))
        if rc != OK:
            raise RuntimeError("oracle_slot_register: %d" % rc)
        self._keep.append(arr)
        return out.value

    def slot_unregister(self, slot: int) -> int:
        return self._lib.oracle_slot_unregister(self._ctx, slot)

    def slot_register_global(self, owner: "Oracle", owner_slot: int):
        """This instance's view of the Global Memory Slot over ``owner``'s local slot.
        Returns (status, slot id)."""
        out = ctypes.c_uint32()
        rc = self._lib.oracle_slot_register_global(self._ctx, owner._ctx, owner_slot, ctypes.byref(out))
        if rc == OK and owner is not self:
            self._keep.append(owner)          # the owner's storage outlives this view
        return rc, (out.value if rc == OK else None)

    def slot_is_global(self, slot: int) -> int:
        """1 = Global Memory Slot, 0 = Local Memory Slot, negative = status."""
        return self._lib.oracle_slot_is_global(self._ctx, slot)

    def slot_global_counters(self, slot: int):
        """Messages of all instances on the Global Memory Slot behind local slot ``slot`` (reading 23)."""
        s, r = ctypes.c_uint64(), ctypes.c_uint64()
        rc = self._lib.oracle_slot_global_counters(self._ctx, slot, ctypes.byref(s), ctypes.byref(r))
        if rc != OK:
            raise RuntimeError("oracle_slot_global_counters: %d" % rc)
        return s.value, r.value

    def slot_counters(self, slot: int):
        s, r = ctypes.c_uint64(), ctypes.c_uint64()
        rc = self._lib.oracle_slot_counters(self._ctx, slot, ctypes.byref(s), ctypes.byref(r))
        if rc != OK:
            raise RuntimeError("oracle_slot_counters: %d" % rc)
        return s.value, r.value

    # -- memcpy / fence ---------------------------------------------------------------
    def memcpy_batch(self, descs: np.ndarray):
        """Returns (status, first_bad).  first_bad is None when status == OK."""
        assert descs.dtype == DESC_DTYPE and descs.flags.c_contiguous
        bad = ctypes.c_uint64(0)
        rc = self._lib.oracle_memcpy_batch(self._ctx, descs.ctypes.data, descs.size, ctypes.byref(bad))
        return rc, (bad.value if rc != OK else None)

    def fence(self) -> int:
        return self._lib.oracle_fence(self._ctx)

    def pending(self) -> int:
        return self._lib.oracle_pending(self._ctx)

    # -- channels -----------------------------------------------------------------------
    def channel_create(self, ring_slot: int, token_bytes: int, capacity: int):
        out = ctypes.c_uint32()
        rc = self._lib.oracle_channel_create(self._ctx, ring_slot, token_bytes, capacity, ctypes.byref(out))
        return rc, (out.value if rc == OK else None)

    def channel_counters(self, ch: int):
        h, t = ctypes.c_uint64(), ctypes.c_uint64()
        rc = self._lib.oracle_channel_counters(self._ctx, ch, ctypes.byref(h), ctypes.byref(t))
        if rc != OK:
            raise RuntimeError("oracle_channel_counters: %d" % rc)
        return h.value, t.value

    def channel_push(self, ch: int, src: int, src_off: int, n: int):
        k = ctypes.c_uint64(0)
        rc = self._lib.oracle_channel_push(self._ctx, ch, src, src_off, n, ctypes.byref(k))
        return rc, k.value

    def channel_pop(self, ch: int, dst: int, dst_off: int, max_n: int):
        k = ctypes.c_uint64(0)
        rc = self._lib.oracle_channel_pop(self._ctx, ch, dst, dst_off, max_n, ctypes.byref(k))
        return rc, k.value
