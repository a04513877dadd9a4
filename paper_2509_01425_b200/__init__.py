"""B200-native HiCR memory-slot copy engine and token channels (arxiv 2509.01425).

The product is the C-ABI library declared in ``include/hicr.h`` and built from
``csrc/*.cu`` for sm_100a; ``binding`` marshals arguments into it (ctypes, and the CPython C
API for the calls of a step).
Importing this package loads (building if stale) ``libhicr_b200.so`` and raises if that
is impossible: there is no CPU fallback and nothing here imports ``oracle/``.
"""
from .binding import (  # noqa: F401
    DESC_DTYPE,
    EXPORTS,
    HICR_ERR_BUSY,
    HICR_ERR_CUDA,
    HICR_ERR_DUPLICATE_KEY,
    HICR_ERR_ILLEGAL_DIRECTION,
    HICR_ERR_INVALID_ARG,
    HICR_ERR_INVALID_SLOT,
    HICR_ERR_NO_CAPACITY,
    HICR_ERR_OUT_OF_BOUNDS,
    HICR_ERR_TIMEOUT,
    HICR_ERR_UNSUPPORTED_SPACE,
    HICR_GLOBAL_HANDLE_BYTES,
    GLOBAL_COUNT_DTYPE,
    HICR_MAX_SLOTS,
    HICR_NOALLOC_MAX_CHUNKS,
    HICR_NOALLOC_MAX_DESCS,
    HICR_NOALLOC_MAX_SLOTS,
    HICR_OK,
    LIB_PATH,
    Channel,
    Context,
    HicrError,
    Mpsc,
    RAW_SLOT_DTYPE,
    lib,
    memcpy_batch_noalloc,
)
from . import collective  # noqa: F401,E402
