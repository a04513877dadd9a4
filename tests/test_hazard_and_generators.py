"""CPU tests for the hazard checker (sweep vs O(n^2) definition) and the seeded generators."""
import numpy as np
import pytest

import workloads as W
from oracle import hazard


def _random_batch(rng, n, n_slots, slot_bytes, max_size):
    d = W.make_descs(rng.integers(0, n_slots, n), rng.integers(0, n_slots, n),
                     np.zeros(n), np.zeros(n), rng.integers(0, max_size + 1, n))
    d["dst_off"] = (rng.random(n) * (slot_bytes - d["size"] + 1)).astype(np.uint64)
    d["src_off"] = (rng.random(n) * (slot_bytes - d["size"] + 1)).astype(np.uint64)
    return d


def test_sweep_equals_bruteforce():
    rng = np.random.default_rng(11)
    seen = {True: 0, False: 0}
    for trial in range(400):
        n = int(rng.integers(1, 7))
        sizes = [64, 64, 64]
        d = _random_batch(rng, n, 3, 64, int(rng.integers(1, 12)))
        ok = hazard.brute_force(d, sizes)
        res = hazard.check(d, sizes)
        assert (res is None) == ok, (d, res)
        seen[ok] += 1
    assert seen[True] > 30 and seen[False] > 30


def test_sweep_named_cases():
    sizes = [32, 32]
    mk = W.make_descs
    assert hazard.check(mk([1, 1], [0, 0], [0, 8], [0, 0], [8, 8]), sizes) is None        # sources may overlap
    assert hazard.check(mk([1, 1], [0, 0], [0, 7], [0, 16], [8, 8]), sizes)[0] == "dst-dst"
    assert hazard.check(mk([0], [0], [4], [0], [8]), sizes)[0] == "dst-src"                # own source
    assert hazard.check(mk([0], [0], [8], [0], [8]), sizes) is None                        # adjacent is fine
    assert hazard.check(mk([0, 1], [1, 0], [0, 0], [0, 4], [8, 8]), sizes)[0] == "dst-src"
    assert hazard.check(mk([0, 0], [1, 1], [0, 0], [0, 0], [0, 8]), sizes) is None         # zero size touches nothing


def test_generators_are_deterministic_and_hazard_free():
    a, b = W.tiny(), W.tiny()
    assert a.epochs[0].tobytes() == b.epochs[0].tobytes()
    assert a.slot_image(0).tobytes() == b.slot_image(0).tobytes()
    assert a.slot_image(0).tobytes() != a.slot_image(1).tobytes()
    assert W.tiny(seed=1).epochs[0].tobytes() != a.epochs[0].tobytes()
    d = a.epochs[0]
    assert len(d) == 256 and d["size"].min() >= 1 and d["size"].max() <= 4096
    assert np.all(d["src_slot"] == 0) and np.all(d["dst_slot"] == 1)
    assert np.all(d["src_off"] + d["size"] <= W.MiB) and np.all(d["dst_off"] + d["size"] <= W.MiB)
    assert hazard.check(d, a.slot_sizes) is None
    assert np.any(d["dst_off"] % 16 != 0) and np.any(d["src_off"] % 16 != 0)  # byte-granular


def test_bulk_aligned_shape():
    w = W.bulk_aligned(n_desc=1024, slot_bytes=32 * W.MiB, n_sets=4)
    allp = np.concatenate([e["dst_off"] for e in w.epochs])
    alls = np.concatenate([e["src_off"] for e in w.epochs])
    assert len(np.unique(allp)) == 4096 and len(np.unique(alls)) == 4096   # sets pairwise disjoint
    for e in w.epochs:
        assert np.all(e["size"] == 4096) and np.all(e["dst_off"] % 4096 == 0) and np.all(e["src_off"] % 4096 == 0)
        assert hazard.check(e, w.slot_sizes) is None


@pytest.mark.parametrize("variant", ["a", "b"])
def test_heavy_tailed_shape(variant):
    w = W.heavy_tailed(variant, n_slots=8, slot_bytes=4 * W.MiB, src_zone=512 * W.KiB, n_desc=3000,
                       smax=256 * W.KiB)
    d = w.epochs[0]
    assert d["size"].min() >= 16 and d["size"].max() <= 256 * W.KiB
    assert np.all(d["src_off"] + d["size"] <= 512 * W.KiB)
    assert np.all(d["dst_off"] >= 512 * W.KiB) and np.all(d["dst_off"] + d["size"] <= 4 * W.MiB)
    assert hazard.check(d, w.slot_sizes) is None
    assert len(np.unique(d["src_slot"])) == 8
    if variant == "b":
        # literal log-uniform: about as many draws per octave
        lg = np.log2(d["size"].astype(float))
        h, _ = np.histogram(lg, bins=[4, 7, 10, 13, 16])
        assert h.min() > 0.5 * h.max()


def test_full_size_config3_numbers_match_survey():
    """the trial draw gave ~10.5 GiB / median 152 B / 2,052 descriptors
    >= 1 MiB for 3a and ~12.4k descriptors / 13.96 GiB for 3b."""
    a = W.heavy_tailed("a")
    assert a.n_descs == 100000 and 10.0 < a.bytes_copied / W.GiB < 11.0
    b = W.heavy_tailed("b")
    assert 11000 < b.n_descs < 14000 and 13.5 < b.bytes_copied / W.GiB <= 14.0
    assert hazard.check(a.epochs[0], a.slot_sizes) is None
    assert hazard.check(b.epochs[0], b.slot_sizes) is None


def test_channel_workloads():
    c = W.spsc(n_tokens=10000, max_batch=100)
    assert c.batches[0].sum() == 10000 and c.batches[0].min() >= 1 and c.batches[0].max() <= 100
    m = W.mpsc(producers=4, n_tokens=500, max_batch=16)
    assert all(b.sum() == 500 for b in m.batches)
    assert np.bincount(m.schedule).tolist() == [len(b) for b in m.batches]
