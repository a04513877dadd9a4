"""Epoch-precondition ("hazard") checker -- TEST INFRASTRUCTURE, part of the oracle.

The paper does not order transfers before the fence ("The completion of a memory transfer
is not guaranteed after the function call returns"), so within one epoch
two transfers that write the same byte, or one that reads what another writes, have no
defined result.  SURVEY.md S8(c) point 5 therefore makes it a PRECONDITION of a batch that

  (1) destination ranges are pairwise disjoint, and
  (2) no destination range overlaps any source range (its own included).

Sources may overlap one another freely; zero-size ranges touch nothing.  This module
checks both by sort-and-sweep in O(n log n) over a flat address space in which slot s
starts at ``bases[s]`` (default: slots laid end to end, i.e. distinct slots are distinct
memory).  ``brute_force`` is the O(n^2) definition the tests pin the sweep against.
"""
from __future__ import annotations

import numpy as np


def _flat(descs, slot_sizes, bases):
    slot_sizes = np.asarray(slot_sizes, dtype=np.uint64)
    if bases is None:
        bases = np.concatenate([[0], np.cumsum(slot_sizes)[:-1]]).astype(np.uint64)
    else:
        bases = np.asarray(bases, dtype=np.uint64)
    size = descs["size"].astype(np.uint64)
    d0 = bases[descs["dst_slot"]] + descs["dst_off"]
    s0 = bases[descs["src_slot"]] + descs["src_off"]
    return d0, s0, size


def check(descs: np.ndarray, slot_sizes, bases=None):
    """Return None if the batch satisfies the precondition, else a tuple
    (kind, i, j): kind 'dst-dst' or 'dst-src', i a destination descriptor index and
    j the index of the descriptor whose destination / source range it overlaps."""
    d0, s0, size = _flat(descs, slot_sizes, bases)
    nz = np.nonzero(size)[0]
    if nz.size == 0:
        return None
    d0, s0, size = d0[nz], s0[nz], size[nz]
    order = np.argsort(d0, kind="stable")
    ds, de = d0[order], d0[order] + size[order]
    # (1) sorted by start, disjoint iff every start >= the previous end
    bad = np.nonzero(ds[1:] < de[:-1])[0]
    if bad.size:
        k = int(bad[0])
        return ("dst-dst", int(nz[order[k + 1]]), int(nz[order[k]]))
    # (2) destinations are now disjoint and sorted, so their ends are sorted too:
    # the first destination whose end exceeds a source's start is the only candidate
    se = s0 + size
    pos = np.searchsorted(de, s0, side="right")
    cand = np.minimum(pos, ds.size - 1)
    hit = (pos < ds.size) & (ds[cand] < se)
    bad = np.nonzero(hit)[0]
    if bad.size:
        k = int(bad[0])
        return ("dst-src", int(nz[order[cand[k]]]), int(nz[k]))
    return None


def brute_force(descs: np.ndarray, slot_sizes, bases=None) -> bool:
    """O(n^2) statement of the precondition; True iff it holds."""
    d0, s0, size = _flat(descs, slot_sizes, bases)
    n = len(descs)
    for i in range(n):
        if size[i] == 0:
            continue
        a0, a1 = int(d0[i]), int(d0[i] + size[i])
        for j in range(n):
            if size[j] == 0:
                continue
            if j != i:
                b0, b1 = int(d0[j]), int(d0[j] + size[j])
                if a0 < b1 and b0 < a1:
                    return False
            c0, c1 = int(s0[j]), int(s0[j] + size[j])
            if a0 < c1 and c0 < a1:
                return False
    return True
