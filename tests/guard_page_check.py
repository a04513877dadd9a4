"""Guard-page check of the copy engine (run as a subprocess by tests/test_gpu_memcpy.py).

Source and destination slots END on the last byte of a mapped 2 MiB granule whose following
virtual addresses are reserved but NOT mapped (CUDA virtual memory management), so any load or
store of the kernels past the end of a slot faults instead of going unnoticed.  Descriptors of
every size class (team, warp, chunk) and alignment end on or near that last byte; the result
is compared with the CPU oracle.  Exit code 0 = no fault, bit-exact.  Test infrastructure.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    import torch
    from cuda.bindings import driver as cu

    import paper_2509_01425_b200 as hicr
    import workloads as W
    from oracle import Oracle

    def ck(res):
        err, *out = res
        if err != cu.CUresult.CUDA_SUCCESS:
            raise RuntimeError("CUDA driver error %s" % err)
        return out[0] if len(out) == 1 else out

    torch.cuda.init()
    torch.zeros(1, device="cuda")                      # primary context current
    prop = cu.CUmemAllocationProp()
    prop.type = cu.CUmemAllocationType.CU_MEM_ALLOCATION_TYPE_PINNED
    prop.location.type = cu.CUmemLocationType.CU_MEM_LOCATION_TYPE_DEVICE
    prop.location.id = 0
    gran = ck(cu.cuMemGetAllocationGranularity(prop, cu.CUmemAllocationGranularity_flags.CU_MEM_ALLOC_GRANULARITY_MINIMUM))
    acc = cu.CUmemAccessDesc()
    acc.location = prop.location
    acc.flags = cu.CUmemAccess_flags.CU_MEM_ACCESS_FLAGS_PROT_READWRITE

    def guarded():
        """gran mapped bytes followed by gran reserved, unmapped bytes; returns the base address."""
        va = int(ck(cu.cuMemAddressReserve(2 * gran, 0, 0, 0)))
        h = ck(cu.cuMemCreate(gran, prop, 0))
        ck(cu.cuMemMap(va, gran, 0, h, 0))
        ck(cu.cuMemSetAccess(va, gran, [acc], 1))
        return va

    src_va, dst_va = guarded(), guarded()
    rng = np.random.default_rng(W.BASE_SEED + 77)
    SLOT = 1 << 20                                      # each slot = the last MiB of its granule
    src_img = rng.integers(0, 256, SLOT, dtype=np.uint8)
    dst_img = rng.integers(0, 256, SLOT, dtype=np.uint8)
    s_base, d_base = src_va + gran - SLOT, dst_va + gran - SLOT
    ck(cu.cuMemcpyHtoD(s_base, src_img.ctypes.data, SLOT))
    ck(cu.cuMemcpyHtoD(d_base, dst_img.ctypes.data, SLOT))

    sizes = list(range(1, 40)) + [63, 64, 65, 127, 128, 129, 255, 256, 257, 300, 1000, 4095, 4096, 4097, 8191, 8192,
                                  8193, 40000, 131072, 131073, 300000, 700001]
    o = Oracle()
    o_src, o_dst = src_img.copy(), dst_img.copy()
    assert o.slot_register(o_src) == 0 and o.slot_register(o_dst) == 1
    ctx = hicr.Context(0, torch.cuda.current_stream().cuda_stream)
    ids = [ctx.slot_register(s_base, SLOT), ctx.slot_register(d_base, SLOT)]
    assert ids == [0, 1]
    n_batches = 0
    for size in sizes:
        for se in (0, 1, 5, 16):                        # bytes between the source range's end and the slot's end
            for de in (0, 3, 16):                       # the same for the destination
                if size + max(se, de) > SLOT:
                    continue
                d = W.make_descs([1], [0], [SLOT - de - size], [SLOT - se - size], [size])
                for device_table in (False, True):
                    assert o.memcpy_batch(d)[0] == 0 and o.fence() == 0
                    if device_table:
                        t = torch.from_numpy(d.view(np.uint8).copy()).cuda()
                        ctx.memcpy_batch(t, n=1)
                    else:
                        ctx.memcpy_batch(d)
                    ctx.fence()
                    n_batches += 1
    # one batch with many descriptors that all read up to the last byte of the source slot
    sz = np.array([s for s in sizes if s <= 4097] * 3, dtype=np.int64)
    dst_off = W.gaps_composition(rng, sz, 0, SLOT - 4)
    dst_off[0] = SLOT - sz[0]                            # and one that writes the last byte of the destination slot
    many = W.make_descs(np.ones(len(sz), np.int64), np.zeros(len(sz), np.int64), dst_off, SLOT - sz, sz)
    keep = np.ones(len(sz), bool)
    keep[1:] = dst_off[1:] + sz[1:] <= SLOT - sz[0]      # keep destinations disjoint from descriptor 0's
    many = np.ascontiguousarray(many[keep])
    assert o.memcpy_batch(many)[0] == 0 and o.fence() == 0
    t = torch.from_numpy(many.view(np.uint8).copy()).cuda()
    ctx.memcpy_batch(t, n=len(many))
    ctx.fence()
    torch.cuda.synchronize()
    got_src, got_dst = np.empty(SLOT, np.uint8), np.empty(SLOT, np.uint8)
    ck(cu.cuMemcpyDtoH(got_src.ctypes.data, s_base, SLOT))
    ck(cu.cuMemcpyDtoH(got_dst.ctypes.data, d_base, SLOT))
    assert got_src.tobytes() == o_src.tobytes() == src_img.tobytes(), "source slot changed"
    assert got_dst.tobytes() == o_dst.tobytes(), "destination slot differs from the oracle"
    assert [ctx.slot_counters(s) for s in ids] == [o.slot_counters(0), o.slot_counters(1)]
    ctx.close()
    print("guard page check ok: %d single-descriptor batches + 1 batch of %d, no fault, bit-exact" % (n_batches, len(many)))
    return 0


if __name__ == "__main__":
    sys.exit(main())
