"""Seeded synthetic inputs for the five BASELINE.json configs (and scaled-down variants).

This module holds NONE of the method's arithmetic: it only draws slot images,
descriptor tables, token streams and push/pop schedules.  The same arrays are handed to
the CPU oracle and to the CUDA library; neither side generates its own inputs.

The paper measures this path on no public dataset; the shapes come from SURVEY.md S8(d)
(which takes them from BASELINE.json's configs and the paper's TC1 size sweep,
PAPER.md:659-661).  Recipe, stated in DESIGN.md "Inputs":

  * base seed 250901425, config c uses PCG64([seed + c, stream]);
  * slot bytes: uniform random uint8;
  * disjoint destinations by *gaps composition*: draw the sizes, slack = region - sum,
    split the slack into n+1 random non-negative gaps, lay the ranges out in a random
    order with those gaps (byte-granular, disjoint, O(n log n)).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 250901425

# 32-byte descriptor, field order = the paper's call memcpy(dst, dst_off, src, src_off, size)
# (PAPER.md:532).  Declared here independently of oracle/ and of include/hicr.h.
DESC_DTYPE = np.dtype(
    [("dst_slot", "<u4"), ("src_slot", "<u4"), ("dst_off", "<u8"), ("src_off", "<u8"), ("size", "<u8")]
)

KiB, MiB, GiB = 1 << 10, 1 << 20, 1 << 30


def rng_for(config: int, stream: int = 0, seed: int = BASE_SEED) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64([seed + config, stream]))


def random_bytes(rng: np.random.Generator, n: int) -> np.ndarray:
    """n uniform random bytes (drawn as 64-bit words; tail from one more word)."""
    words = (n + 7) // 8
    b = rng.integers(0, 1 << 64, size=words, dtype=np.uint64).view(np.uint8)
    return b if n % 8 == 0 else b[:n].copy()


def gaps_composition(rng: np.random.Generator, sizes: np.ndarray, lo: int, hi: int) -> np.ndarray:
    """Offsets in [lo, hi) for ranges of the given sizes: pairwise disjoint, random order,
    random gaps.  Returns offsets in the order of ``sizes``.  Raises if they do not fit."""
    sizes = np.asarray(sizes, dtype=np.int64)
    n = sizes.size
    total = int(sizes.sum())
    slack = (hi - lo) - total
    if slack < 0:
        raise ValueError("ranges of total size %d do not fit a region of %d" % (total, hi - lo))
    if n == 0:
        return np.zeros(0, dtype=np.uint64)
    # n+1 non-negative gaps summing to slack: n sorted cut points in [0, slack]
    cuts = np.sort(rng.integers(0, slack + 1, size=n, dtype=np.int64))
    gaps = np.diff(np.concatenate([[0], cuts]))  # gap before each range; last gap is implicit
    order = rng.permutation(n)  # order[k] = which descriptor sits k-th in the region
    laid = sizes[order]
    starts = lo + np.cumsum(gaps) + np.concatenate([[0], np.cumsum(laid)[:-1]])
    out = np.empty(n, dtype=np.uint64)
    out[order] = starts.astype(np.uint64)
    return out


def make_descs(dst_slot, src_slot, dst_off, src_off, size) -> np.ndarray:
    n = len(size)
    d = np.zeros(n, dtype=DESC_DTYPE)
    d["dst_slot"] = dst_slot
    d["src_slot"] = src_slot
    d["dst_off"] = dst_off
    d["src_off"] = src_off
    d["size"] = size
    return d


@dataclass
class CopyWorkload:
    """slot_sizes[s] bytes per slot; slot images are drawn by ``slot_image(s)`` on demand
    (so a 16 GiB config never has to be held twice); epochs = list of descriptor tables,
    one fence after each."""
    name: str
    config: int
    slot_sizes: list
    epochs: list
    seed: int = BASE_SEED
    meta: dict = field(default_factory=dict)

    def slot_image(self, s: int) -> np.ndarray:
        return random_bytes(rng_for(self.config, 1000 + s, self.seed), int(self.slot_sizes[s]))

    @property
    def n_descs(self) -> int:
        return int(sum(len(e) for e in self.epochs))

    @property
    def bytes_copied(self) -> int:
        return int(sum(int(e["size"].sum()) for e in self.epochs))


# ---------------------------------------------------------------------------------- C1
def tiny(n_desc: int = 256, slot_bytes: int = MiB, max_size: int = 4096, seed: int = BASE_SEED) -> CopyWorkload:
    """Config 1: 2 slots; n_desc descriptors slot 0 -> slot 1; size ~ U{1..max_size};
    byte-granular src offsets; destinations by gaps composition over slot 1; 1 fence."""
    rng = rng_for(1, 0, seed)
    size = rng.integers(1, max_size + 1, size=n_desc, dtype=np.int64)
    src_off = (rng.random(n_desc) * (slot_bytes - size + 1)).astype(np.int64)
    src_off = np.minimum(src_off, slot_bytes - size)
    dst_off = gaps_composition(rng, size, 0, slot_bytes)
    d = make_descs(1, 0, dst_off, src_off, size)
    return CopyWorkload("tiny", 1, [slot_bytes, slot_bytes], [d], seed)


# ---------------------------------------------------------------------------------- C2
def bulk_aligned(n_desc: int = 65536, slot_bytes: int = GiB, page: int = 4096, n_sets: int = 4,
                 seed: int = BASE_SEED) -> CopyWorkload:
    """Config 2: 2 slots; n_desc descriptors of exactly ``page`` bytes at page-aligned
    offsets; destination pages a random sample without replacement of slot 1's pages,
    source pages likewise of slot 0's (reading 20).  ``n_sets`` pairwise-disjoint
    descriptor sets are returned as ``epochs`` (one fence each); bench.py rotates through
    them so that 1.5 GiB of other traffic separates reuse of a page (cold L2)."""
    rng = rng_for(2, 0, seed)
    n_pages = slot_bytes // page
    if n_sets * n_desc > n_pages:
        raise ValueError("not enough pages for %d disjoint sets" % n_sets)
    dpages = rng.permutation(n_pages)[: n_sets * n_desc].astype(np.int64)
    spages = rng.permutation(n_pages)[: n_sets * n_desc].astype(np.int64)
    epochs = []
    for k in range(n_sets):
        sl = slice(k * n_desc, (k + 1) * n_desc)
        epochs.append(make_descs(1, 0, dpages[sl] * page, spages[sl] * page, np.full(n_desc, page)))
    return CopyWorkload("bulk_aligned", 2, [slot_bytes, slot_bytes], epochs, seed, {"page": page})


# ---------------------------------------------------------------------------------- C3
def _power_law_sizes(rng, n, a, b, alpha):
    """Inverse CDF of p(s) ~ s^-alpha on [a, b]; alpha = 1 is the log-uniform law."""
    u = rng.random(n)
    if abs(alpha - 1.0) < 1e-12:
        s = a * (b / a) ** u
    else:
        e = 1.0 - alpha
        s = (a ** e + u * (b ** e - a ** e)) ** (1.0 / e)
    return np.clip(np.floor(s).astype(np.int64), a, b)


def heavy_tailed(variant: str = "a", n_slots: int = 64, slot_bytes: int = 256 * MiB,
                 src_zone: int = 32 * MiB, n_desc: int = 100000, smin: int = 16, smax: int = 16 * MiB,
                 alpha: float = 1.3, seed: int = BASE_SEED, align: int = 1) -> CopyWorkload:
    """Config 3 (reading 19: BASELINE.json's literal text needs 112.7 GiB of disjoint
    destinations inside 16 GiB, so two variants are run).

    Every slot: bytes [0, src_zone) are the source zone, [src_zone, slot_bytes) the
    destination zone, so no destination overlaps any source.  src_slot ~ U; dst_slot
    uniform among the slots whose remaining destination room >= size; src_off uniform in
    the source zone; dst_off by gaps composition per slot; all byte-granular.

      'a': n_desc sizes from the truncated power law p(s) ~ s^-alpha on [smin, smax].
      'b': literal log-uniform sizes floor(smin * 2^(log2(smax/smin) u)), taken in draw
           order until no slot has room for the next one (at most n_desc).

    ``align`` > 1 (not a BASELINE config; used to measure the bulk-copy path): offsets and sizes
    rounded DOWN to multiples of ``align`` afterwards, which keeps the ranges disjoint."""
    rng = rng_for(3, 0 if variant == "a" else 1, seed)
    room = np.full(n_slots, slot_bytes - src_zone, dtype=np.int64)
    if variant == "a":
        size = _power_law_sizes(rng, n_desc, smin, smax, alpha)
    elif variant == "b":
        size = _power_law_sizes(rng, n_desc, smin, smax, 1.0)
    else:
        raise ValueError(variant)
    pick = rng.random(n_desc)
    dst_slot = np.empty(n_desc, dtype=np.int64)
    n_used = n_desc
    for i in range(n_desc):
        ok = np.nonzero(room >= size[i])[0]
        if ok.size == 0:
            if variant == "b":
                n_used = i
                break
            raise ValueError("descriptor %d of %d bytes fits no slot" % (i, size[i]))
        s = ok[min(int(pick[i] * ok.size), ok.size - 1)]
        dst_slot[i] = s
        room[s] -= size[i]
    size, dst_slot = size[:n_used], dst_slot[:n_used]
    src_slot = rng.integers(0, n_slots, size=n_used, dtype=np.int64)
    src_off = np.minimum((rng.random(n_used) * (src_zone - size + 1)).astype(np.int64), src_zone - size)
    dst_off = np.zeros(n_used, dtype=np.uint64)
    for s in range(n_slots):
        idx = np.nonzero(dst_slot == s)[0]
        dst_off[idx] = gaps_composition(rng, size[idx], src_zone, slot_bytes)
    if align > 1:
        size = np.maximum(size // align * align, align)
        src_off = src_off // align * align
        dst_off = dst_off // np.uint64(align) * np.uint64(align)
    d = make_descs(dst_slot, src_slot, dst_off, src_off, size)
    return CopyWorkload("heavy_tailed_3" + variant + ("_aligned%d" % align if align > 1 else ""), 3, [slot_bytes] * n_slots, [d], seed,
                        {"variant": variant, "alpha": alpha if variant == "a" else 1.0, "src_zone": src_zone})


# ---------------------------------------------------------------------------------- C4
def chained_epochs(n_epochs: int = 64, n_desc: int = 65536, slot_bytes: int = 256 * MiB,
                   smin: int = 8, smax: int = 256, seed: int = BASE_SEED) -> CopyWorkload:
    """Config 4: one slot split into halves A = [0, H) and B = [H, 2H).  Epoch k writes
    into B if k is even, A if odd, and reads from the other half.  size ~ U{smin..smax};
    destinations by gaps composition in the target half.  Epoch 0 sources: uniform in A.
    Epoch k+1 sources (reading 22): draw the size, pick a parent uniformly among epoch-k
    descriptors with size >= it (clamp the size to the largest parent if none),
    sub-offset uniform inside the parent's destination range.  One fence per epoch."""
    rng = rng_for(4, 0, seed)
    H = slot_bytes // 2
    epochs = []
    prev = None
    for k in range(n_epochs):
        wlo = H if k % 2 == 0 else 0
        rlo = 0 if k % 2 == 0 else H
        size = rng.integers(smin, smax + 1, size=n_desc, dtype=np.int64)
        if prev is None:
            src_off = rlo + np.minimum((rng.random(n_desc) * (H - size + 1)).astype(np.int64), H - size)
        else:
            psize = prev["size"].astype(np.int64)
            order = np.argsort(psize, kind="stable")
            sorted_sizes = psize[order]
            size = np.minimum(size, sorted_sizes[-1])
            pos = np.searchsorted(sorted_sizes, size, side="left")  # parents order[pos:] have size >= it
            u = rng.random(n_desc)
            parent = order[np.minimum(pos + (u * (n_desc - pos)).astype(np.int64), n_desc - 1)]
            sub = np.minimum((rng.random(n_desc) * (psize[parent] - size + 1)).astype(np.int64),
                             psize[parent] - size)
            src_off = prev["dst_off"][parent].astype(np.int64) + sub
        dst_off = gaps_composition(rng, size, wlo, wlo + H)
        d = make_descs(0, 0, dst_off, src_off, size)
        epochs.append(d)
        prev = d
    return CopyWorkload("chained_epochs", 4, [slot_bytes], epochs, seed)


# ---------------------------------------------------------------------------------- C5
@dataclass
class ChannelWorkload:
    """SPSC / non-locking MPSC token streams.  producers P, token_bytes T, capacity C,
    n_tokens per producer.  ``batches[p]`` = push sizes of producer p (sum = n_tokens).
    ``schedule`` (MPSC only) = int array of producer ids: the seeded order in which the
    harness lets producers push their next batch (the consumer drains that ring right
    after, reading 13)."""
    name: str
    producers: int
    token_bytes: int
    capacity: int
    n_tokens: int
    batches: list
    schedule: np.ndarray
    seed: int = BASE_SEED

    def source_image(self, p: int) -> np.ndarray:
        return random_bytes(rng_for(5, 1000 + p, self.seed), self.n_tokens * self.token_bytes)


def _batches(rng, n_tokens, max_batch):
    out = []
    left = n_tokens
    while left > 0:
        draw = rng.integers(1, max_batch + 1, size=max(16, 2 * left // max_batch + 16), dtype=np.int64)
        for b in draw:
            b = int(min(b, left))
            out.append(b)
            left -= b
            if left == 0:
                break
    return np.asarray(out, dtype=np.int64)


def spsc(n_tokens: int = 1 << 24, token_bytes: int = 256, capacity: int = 1024, max_batch: int = 1024,
         seed: int = BASE_SEED) -> ChannelWorkload:
    """Config 5a: batch sizes ~ U{1..max_batch} until they sum to n_tokens (last clipped);
    loop push(b_i) then pop(max = capacity)."""
    rng = rng_for(5, 0, seed)
    b = _batches(rng, n_tokens, max_batch)
    return ChannelWorkload("spsc", 1, token_bytes, capacity, n_tokens, [b], np.zeros(len(b), dtype=np.int64), seed)


def mpsc(producers: int = 148, n_tokens: int = 1 << 20, token_bytes: int = 64, capacity: int = 1024,
         max_batch: int = 256, seed: int = BASE_SEED) -> ChannelWorkload:
    """Config 5b (readings 16-18): non-locking MPSC = one ring per producer; producer p
    pushes batches ~ U{1..max_batch}; ``schedule`` is a seeded shuffle of all producers'
    batch slots, i.e. the order in which the oracle interleaves them."""
    rng = rng_for(5, 1, seed)
    batches = [_batches(rng, n_tokens, max_batch) for _ in range(producers)]
    sched = np.concatenate([np.full(len(b), p, dtype=np.int64) for p, b in enumerate(batches)])
    rng.shuffle(sched)
    return ChannelWorkload("mpsc", producers, token_bytes, capacity, n_tokens, batches, sched, seed)


def tagged_sources(producers: int, n_tokens: int, token_bytes: int, seed: int = BASE_SEED):
    """Sources for the LOCKING MPSC run, whose interleaving in the sink is
    not defined: token i of producer p is random bytes with a tag in its first 8 bytes --
    little-endian u32 p, u32 i -- so that a checker can recover, from the sink alone, which
    producer's which token sits where (per-producer order, every token exactly once)."""
    if token_bytes < 8:
        raise ValueError("tagged tokens need at least 8 bytes")
    out = []
    for p in range(producers):
        a = random_bytes(rng_for(5, 2000 + p, seed), n_tokens * token_bytes).reshape(n_tokens, token_bytes)
        tag = np.empty((n_tokens, 2), dtype="<u4")
        tag[:, 0] = p
        tag[:, 1] = np.arange(n_tokens, dtype=np.uint32)
        a[:, :8] = tag.view(np.uint8).reshape(n_tokens, 8)
        out.append(np.ascontiguousarray(a.reshape(-1)))
    return out


# ---------------------------------------------------------------------------------- global slots
@dataclass
class GlobalWorkload:
    """A copy graph over several instances ("randomized
    copy-graph").  Every instance has four buffers: ``lsrc`` / ``ldst`` stay local, ``gsrc`` /
    ``gdst`` are volunteered under ``tag`` with keys 2 i and 2 i + 1.  ``plans[i]`` lists the
    transfers instance i initiates as (dst, dst_off, src, src_off, size) with dst / src =
    ("L", name) for one of its own local buffers or ("G", key) for a global slot.  Sources are
    only read and destinations only written, destination ranges are pairwise disjoint over ALL
    instances (the epoch precondition of reading 5, extended to the global epoch), and no
    transfer names two global slots."""
    n_instances: int
    tag: int
    sizes: dict
    plans: list
    seed: int

    def image(self, instance: int, name: str) -> np.ndarray:
        return random_bytes(rng_for(6, 100 * instance + ("lsrc", "ldst", "gsrc", "gdst").index(name), self.seed),
                            self.sizes[name])


def global_copy_graph(n_instances: int = 2, per_buffer: int = 12, src_bytes: int = 4096, dst_bytes: int = 65536,
                      max_size: int = 3000, seed: int = BASE_SEED, tag: int = 3) -> GlobalWorkload:
    """Local-to-Local, Local-to-Global (put) and Global-to-Local (get) transfers dealt to random
    initiators; sizes uniform in 0..max_size (zero-size transfers included), byte-granular offsets,
    destinations by gaps composition."""
    rng = rng_for(6, 0, seed + n_instances)
    plans = [[] for _ in range(n_instances)]
    for owner in range(n_instances):
        for kind in ("ldst", "gdst"):
            sizes = rng.integers(0, max_size + 1, size=per_buffer)
            offs = gaps_composition(rng, sizes, 0, dst_bytes)
            for sz, off in zip(sizes, offs):
                sz, off = int(sz), int(off)
                if kind == "ldst":
                    init = owner                                     # a local slot is reachable by its instance only
                    dst = ("L", "ldst")
                    src_owner = int(rng.integers(0, n_instances))
                    src = ("L", "lsrc") if (src_owner == init and rng.random() < 0.5) else ("G", 2 * src_owner)
                else:
                    init = int(rng.integers(0, n_instances))         # anyone may put into a global slot
                    dst = ("G", 2 * owner + 1)
                    src = ("L", "lsrc")
                so = int(rng.integers(0, src_bytes - min(sz, src_bytes) + 1))
                plans[init].append((dst, off, src, so, min(sz, src_bytes)))
    for p in plans:
        order = rng.permutation(len(p))
        p[:] = [p[j] for j in order]
    sizes = {"lsrc": src_bytes, "ldst": dst_bytes, "gsrc": src_bytes, "gdst": dst_bytes}
    return GlobalWorkload(n_instances, tag, sizes, plans, seed)
