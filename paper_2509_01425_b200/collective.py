"""Control plane of the Global Memory Slots: carries the library's opaque byte blobs between
instances, nothing else.

The C-ABI library has no transport of its own (include/hicr.h): the collective exchange of
PAPER.md:377-379 and the count exchange of the global fence are each split
into local halves, and this module moves the bytes of one half to the other:

  * ``exchange_global_slots`` / ``fence_global``: one process per instance, the blobs travel by
    ``torch.distributed.all_gather_object`` over whatever backend the group has (gloo or nccl);
  * ``exchange_in_process`` / ``fence_in_process``: several contexts of ONE process standing for
    several instances (tests, single-process multi-GPU), the blobs travel by a Python list.

No slot byte and no counter arithmetic is touched here: the handles are built and consumed by
hicr_global_volunteer / hicr_global_exchange, the counts by hicr_global_fence_begin / _end.
The order all instances agree on is: by instance rank, then by the order the instance listed
its contributions.
"""
from __future__ import annotations

import numpy as np

from .binding import GLOBAL_COUNT_DTYPE, Context


def _all_gather(obj, group=None):
    import torch.distributed as dist
    out = [None] * dist.get_world_size(group)
    dist.all_gather_object(out, obj, group=group)
    return out


def exchange_global_slots(ctx: Context, tag: int, contributions, group=None) -> dict:
    """Collective over ``group``: ``contributions`` = list of (key, local slot) this instance
    volunteers under ``tag`` (may be empty: "volunteering zero or more").  Returns
    {key: global slot id in ``ctx``} for the contributions of ALL instances."""
    mine = [(int(k), ctx.global_volunteer(tag, int(k), int(s))) for k, s in contributions]
    everyone = _all_gather(mine, group)
    keys = [k for inst in everyone for k, _ in inst]
    ids = ctx.global_exchange(tag, [h for inst in everyone for _, h in inst])
    return dict(zip(keys, ids))


def fence_global(ctx: Context, group=None, timeout_ms: int = 0) -> None:
    """Collective global fence: this instance's transfers are complete (blocking local fence),
    every instance tells every other what it initiated on each global slot, and each owner waits
    until its device-side totals have reached the sums ("the expected number of
    incoming and outgoing data transfers")."""
    mine, deferred = ctx.global_fence_begin(defer_error=True)
    everyone = _all_gather(mine.tobytes(), group)                 # (a rank with a rejected batch still takes part)
    ctx.global_fence_end(np.frombuffer(b"".join(everyone), dtype=GLOBAL_COUNT_DTYPE), timeout_ms)
    if deferred is not None:
        raise deferred


def exchange_in_process(ctxs, tag: int, contributions) -> list:
    """The same exchange between contexts of this process: ``contributions[i]`` belongs to
    ``ctxs[i]``.  Returns one {key: global slot id} per context."""
    everyone = [[(int(k), c.global_volunteer(tag, int(k), int(s))) for k, s in contrib]
                for c, contrib in zip(ctxs, contributions)]
    keys = [k for inst in everyone for k, _ in inst]
    handles = [h for inst in everyone for _, h in inst]
    return [dict(zip(keys, c.global_exchange(tag, handles))) for c in ctxs]


def fence_in_process(ctxs, timeout_ms: int = 0) -> None:
    got = [c.global_fence_begin(defer_error=True) for c in ctxs]
    everyone = np.concatenate([g[0] for g in got]) if got else np.zeros(0, dtype=GLOBAL_COUNT_DTYPE)
    for c in ctxs:
        c.global_fence_end(everyone, timeout_ms)
    for _, deferred in got:
        if deferred is not None:
            raise deferred
