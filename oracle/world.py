"""Several HiCR instances in one process, for the oracle (TEST INFRASTRUCTURE, like the rest of
``oracle/``): the collective exchange of Global Memory Slots and the fence over all instances.

PAPER.md:377-379 (S3.1.4): "The exchange of global memory slots is a collective operation: all
instances must participate by volunteering zero or more local memory slots.  The operation
returns as many global memory slots as the total amount of local memory slots exchanged.  Each
of the resulting global memory slots are uniquely identified by a tag and key pair".

An instance is one ``Oracle`` context (hicr_oracle.c); a Global Memory Slot is, in every
instance's table, a slot of kind GLOBAL over the storage of the owner's volunteered local slot
(``oracle_slot_register_global``).  The byte loops, the direction rule and the counters are in
hicr_oracle.c; this module only keeps the (tag, key) bookkeeping of the exchange, written in
the order the paper states it.

Readings (S2, 23-26; the paper fixes none of them):
  * keys are caller-chosen and unique within a tag over ALL instances; a repeated (tag, key)
    fails the whole exchange on every instance ("DuplicateKey") and creates nothing;
  * every instance receives the same set of global slots, its own contributions included, in
    one agreed order: by instance, then by the order the instance listed them;
  * an instance may take part in several exchanges (different tags);
  * the global fence is "every instance fences": after it every transfer any instance
    initiated is complete, and the owner's global counters of a slot equal the sum over all
    instances of their own counts on it.
"""
from __future__ import annotations

from . import ERR_DUPLICATE_KEY, ERR_INVALID_ARG, ERR_INVALID_SLOT, OK, Oracle


class World:
    """``n`` instances, each an ``Oracle``."""

    def __init__(self, n: int):
        self.inst = [Oracle() for _ in range(n)]
        self.table = {}    # (tag, key) -> (owner instance, owner's local slot, [global slot id per instance])

    def exchange(self, tag: int, contributions):
        """``contributions[i]`` = list of (key, local slot of instance i).  Returns (status,
        per-instance dict key -> global slot id).  All-or-nothing."""
        assert len(contributions) == len(self.inst)            # collective: every instance takes part
        seen = set()
        for i, contrib in enumerate(contributions):
            for key, slot in contrib:
                if (tag, key) in self.table or key in seen:
                    return ERR_DUPLICATE_KEY, None
                seen.add(key)
                kind = self.inst[i].slot_is_global(slot)       # a registered LOCAL slot of that instance:
                if kind < 0:                                   # "volunteering zero or more local memory slots"
                    return ERR_INVALID_SLOT, None
                if kind != 0:
                    return ERR_INVALID_ARG, None
        out = [dict() for _ in self.inst]
        for i, contrib in enumerate(contributions):            # by instance, then in the order listed
            for key, slot in contrib:
                ids = []
                for j, o in enumerate(self.inst):
                    rc, g = o.slot_register_global(self.inst[i], slot)
                    assert rc == OK
                    ids.append(g)
                    out[j][key] = g
                self.table[(tag, key)] = (i, slot, ids)
        return OK, out

    def lookup(self, instance: int, tag: int, key: int):
        """getGlobalSlot: the id of (tag, key) in ``instance``'s table, or None."""
        e = self.table.get((tag, key))
        return None if e is None else e[2][instance]

    def fence_all(self):
        """Every instance fences (each closes its own epoch)."""
        return [o.fence() for o in self.inst]
