"""Shared by the Global Memory Slot tests: the same copy graph set up on the oracle's World and on
a set of CUDA contexts (one per instance), and the comparison of everything observable."""
import numpy as np

import oracle
import workloads as W
from oracle.world import World

NAMES = ("lsrc", "ldst", "gsrc", "gdst")


def oracle_run(w):
    """The oracle's result for the workload: (world, images [instance][name], local ids, global ids)."""
    world = World(w.n_instances)
    mem = [{k: w.image(i, k) for k in NAMES} for i in range(w.n_instances)]
    ids = [{k: world.inst[i].slot_register(mem[i][k]) for k in NAMES} for i in range(w.n_instances)]
    rc, g = world.exchange(w.tag, [[(2 * i, ids[i]["gsrc"]), (2 * i + 1, ids[i]["gdst"])] for i in range(w.n_instances)])
    assert rc == oracle.OK
    for i in range(w.n_instances):
        d = descs_for(w, i, ids[i], g[i])
        rc, bad = world.inst[i].memcpy_batch(d)
        assert rc == oracle.OK, (rc, bad)
    assert world.fence_all() == [oracle.OK] * w.n_instances
    return world, mem, ids, g


def descs_for(w, i, local_ids, global_ids):
    """Instance i's descriptor table: ("L", name) -> its local id, ("G", key) -> its id of that global slot."""
    ref = lambda r: local_ids[r[1]] if r[0] == "L" else global_ids[r[1]]
    p = w.plans[i]
    return W.make_descs([ref(t[0]) for t in p], [ref(t[2]) for t in p], [t[1] for t in p], [t[3] for t in p],
                        [t[4] for t in p])
