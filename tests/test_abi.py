"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol that
include/hicr.h declares, the binding's constants and descriptor layout match the header,
and the product path fails loudly without a CUDA device (no CPU fallback, no oracle)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "hicr.h")


def _declared():
    text = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)
    return sorted(set(re.findall(r"\b(hicr_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_2509_01425_b200 as hicr
    names = _declared()
    assert len(names) >= 20 and {"hicr_slot_register", "hicr_memcpy_batch", "hicr_fence", "hicr_channel_push",
                                 "hicr_channel_pop"} <= set(names)
    raw = ctypes.CDLL(hicr.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), "libhicr_b200.so does not export %s" % n
    assert sorted(hicr.EXPORTS) == names


def test_constants_and_descriptor_layout_match_header():
    import paper_2509_01425_b200 as hicr
    text = open(HEADER).read()
    for name in ("HICR_OK", "HICR_ERR_INVALID_ARG", "HICR_ERR_INVALID_SLOT", "HICR_ERR_OUT_OF_BOUNDS",
                 "HICR_ERR_UNSUPPORTED_SPACE", "HICR_ERR_NO_CAPACITY", "HICR_ERR_CUDA", "HICR_ERR_BUSY"):
        m = re.search(r"#define\s+%s\s+\(?(-?\d+)\)?" % name, text)
        assert m and int(m.group(1)) == getattr(hicr, name), name
    assert int(re.search(r"#define\s+HICR_MAX_SLOTS\s+(\d+)u", text).group(1)) == hicr.HICR_MAX_SLOTS
    # field order dst_slot, src_slot, dst_off, src_off, size = the paper's call
    body = re.search(r"typedef struct hicr_desc \{(.*?)\} hicr_desc_t;", text, flags=re.S).group(1)
    fields = re.findall(r"uint(32|64)_t\s+(\w+);", body)
    assert [f[1] for f in fields] == list(hicr.DESC_DTYPE.names)
    assert sum(int(f[0]) // 8 for f in fields) == hicr.DESC_DTYPE.itemsize == 32
    import workloads
    assert workloads.DESC_DTYPE == hicr.DESC_DTYPE


def test_status_text():
    import paper_2509_01425_b200 as hicr
    assert hicr.lib.hicr_strerror(hicr.HICR_OK) == b"ok"
    assert b"slot" in hicr.lib.hicr_strerror(hicr.HICR_ERR_INVALID_SLOT)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2509_01425_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no oracle", "").replace('imports ``oracle/``', ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2509_01425_b200" not in src and "hicr.h" not in src.replace("include/hicr.h", "")


def test_fails_loudly_without_a_gpu():
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_2509_01425_b200 as hicr
    with pytest.raises(hicr.HicrError) as e:
        hicr.Context(0, 0)
    assert e.value.status == hicr.HICR_ERR_CUDA
    # NULL arguments are rejected before any device work
    assert hicr.lib.hicr_fence(None) == hicr.HICR_ERR_INVALID_ARG
    assert hicr.lib.hicr_memcpy_batch(None, None, 0, 0, None) == hicr.HICR_ERR_INVALID_ARG


def test_noalloc_entry_point_refuses_on_the_host_what_it_can():
    """hicr_memcpy_batch_noalloc checks its limits and its pointers before it touches CUDA, so a
    caller learns about a batch that cannot fit the fixed scratch array without a device, and the
    binding's limits are the header's."""
    import paper_2509_01425_b200 as hicr
    text = open(HEADER).read()
    for name in ("HICR_NOALLOC_MAX_DESCS", "HICR_NOALLOC_MAX_SLOTS", "HICR_NOALLOC_MAX_CHUNKS"):
        assert int(re.search(r"#define\s+%s\s+(\d+)u" % name, text).group(1)) == getattr(hicr, name), name
    body = re.search(r"typedef struct hicr_raw_slot \{(.*?)\} hicr_raw_slot_t;", text, flags=re.S).group(1)
    assert re.findall(r"(\w+);", body) == list(hicr.RAW_SLOT_DTYPE.names) and hicr.RAW_SLOT_DTYPE.itemsize == 16
    call = hicr.lib.hicr_memcpy_batch_noalloc
    p = 0x1000          # never dereferenced: every case below is refused first
    assert call(0, None, p, 2, p, hicr.HICR_NOALLOC_MAX_DESCS + 1, p, p) == hicr.HICR_ERR_NO_CAPACITY
    assert call(0, None, p, hicr.HICR_NOALLOC_MAX_SLOTS + 1, p, 1, p, p) == hicr.HICR_ERR_NO_CAPACITY
    assert call(0, None, p, 2, p, 1, p, None) == hicr.HICR_ERR_INVALID_ARG      # no result words
    assert call(0, None, None, 2, p, 1, p, p) == hicr.HICR_ERR_INVALID_ARG      # slots promised, none given
    assert call(0, None, p, 2, None, 1, p, p) == hicr.HICR_ERR_INVALID_ARG      # descriptors promised, none given
    assert call(-1, None, p, 2, p, 1, p, p) == hicr.HICR_ERR_INVALID_ARG
    with pytest.raises(hicr.HicrError) as e:
        hicr.memcpy_batch_noalloc(0, 0, p, 2, p, hicr.HICR_NOALLOC_MAX_DESCS + 1, p, p)
    assert e.value.status == hicr.HICR_ERR_NO_CAPACITY
