#!/usr/bin/env python
"""bench.py -- times the hot path of the B200 HiCR copy engine and prints ONE JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config NAME] [--impl reference]

A *step* is one pass of the whole hot path over one batch of synthetic input:
``hicr_memcpy_batch`` (descriptor ingest + validation, binning, copy kernels, counter
accumulation) followed by ``hicr_fence``.  The default workload is BASELINE.json's
config 2 ("bulk aligned": 2 slots x 1 GiB, 65,536 descriptors of 4 KiB per step, four
pairwise-disjoint descriptor sets rotated so a page is re-touched only after 2 GiB of
other traffic).  ``metric`` = effective GB/s = (bytes read + bytes written) / time.

  value        device-resident descriptor tables, inputs in HBM when timing starts
  e2e          the same call with HOST descriptor tables (the step's input) copied to
               the device inside the timed region and the fence's counter read-back
  roofline     dominant copy kernel, CUDA events recorded by the library around it
  cpu_baseline the CPU oracle (oracle/, as it stands) on the host cores, same workload

N > 1 (torchrun): the path shards by slot ownership with no data-path collective -- every
rank owns its own slots and descriptor sets (seed + rank); weak scaling; the time is the
max over ranks.  ``--impl reference`` times the oracle instead (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC = "memory-slot memcpy effective GB/s (read+write)"
UNIT = "GB/s"


# --------------------------------------------------------------------------- workloads
def make_workload(name: str, rank: int = 0):
    seed = W.BASE_SEED + 1000 * rank
    if name == "bulk":
        return W.bulk_aligned(seed=seed)
    if name == "bulk_small":            # CPU-sized stand-in used by the tests of this file
        return W.bulk_aligned(n_desc=1024, slot_bytes=32 * W.MiB, n_sets=4, seed=seed)
    if name == "tiny":
        return W.tiny(seed=seed)
    if name == "heavy_a":
        return W.heavy_tailed("a", seed=seed)
    if name == "heavy_b":
        return W.heavy_tailed("b", seed=seed)
    if name == "heavy_b_aligned":
        return W.heavy_tailed("b", seed=seed, align=16)
    if name in ("chain", "chain_async", "chain_graph"):
        return W.chained_epochs(seed=seed)
    raise SystemExit("unknown --config %s" % name)


WORKLOAD_TEXT = {
    "bulk": "config 2 bulk aligned: 2 slots x 1 GiB, 65536 x 4 KiB descriptors per step, 4 KiB-aligned, "
            "random page permutation, 1 fence per step",
    "bulk_small": "config 2 scaled down (test only)",
    "tiny": "config 1 tiny: 2 slots x 1 MiB, 256 descriptors of 1..4096 B, 1 fence per step",
    "heavy_a": "config 3a heavy-tailed: 64 slots x 256 MiB, 100000 descriptors, power law 1.3 on 16 B..16 MiB",
    "heavy_b": "config 3b heavy-tailed: 64 slots x 256 MiB, log-uniform 16 B..16 MiB until full",
    "heavy_b_aligned": "config 3b with offsets and sizes rounded down to multiples of 16 B (NOT a BASELINE config: every "
                       "chunk is eligible for the bulk-copy path; run with HICR_TMA_MIN=0xffffffff for the vector path)",
    "chain": "config 4 chained epochs: 1 slot x 256 MiB, 64 epochs x 65536 descriptors of 8..256 B",
    "chain_async": "config 4 chained epochs with stream-ordered fences (hicr_fence_async) between epochs and ONE blocking "
                   "fence at the end of the timed region (SURVEY.md S8(f) 3)",
    "chain_graph": "config 4 chained epochs recorded once as ONE CUDA graph of 64 batches (hicr_graph_*) and replayed: one "
                   "call enqueues 64 epochs, one blocking fence per replay; every replay validates, bins, copies and counts "
                   "on the device (SURVEY.md S8(f) 3)",
}


def shard_report(per_rank_bytes, per_rank_descs, elapsed_ms_max, steps):
    """Whole-job aggregate over ranks (weak scaling, no data-path collective): all ranks'
    units over the slowest rank's time."""
    secs = elapsed_ms_max / 1e3
    return {
        "value": float(sum(per_rank_bytes)) / secs / 1e9,
        "descs_per_s": float(sum(per_rank_descs)) / secs,
        "ms_per_step": elapsed_ms_max / steps,
    }


def rank_max(x: float, dist=None, device="cpu") -> float:
    """Max over ranks of a per-rank time (the job's time is the slowest rank's)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed legs run -- in a process
    of its own: a sampling THREAD takes the interpreter lock for tens of microseconds per sample,
    which a 2 ms timed region of 100 us steps pays for (5 us per step at 20 steps).  The child
    stamps every sample with the wall clock; the parent keeps those that fall into its windows."""

    REASONS = {
        0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
        0x80: "hw_power_brake", 0x2: "applications_clocks", 0x100: "display_clock", 0x10: "sync_boost",
    }
    CHILD = r"""
import sys, time
import pynvml as nv
nv.nvmlInit()
h = nv.nvmlDeviceGetHandleByIndex(int(sys.argv[1]))
period = float(sys.argv[2])
def reasons():
    try:
        return int(nv.nvmlDeviceGetCurrentClocksEventReasons(h))
    except Exception:
        try:
            return int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
        except Exception:
            return 0
for _ in range(3):                      # the first queries of a process take milliseconds: have them behind us
    reasons(); nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
print("max %d" % nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM), flush=True)
while True:
    print("%.6f %d %d" % (time.time(), nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM), reasons()), flush=True)
    time.sleep(period)
"""

    def __init__(self, index: int, period_s: float = 0.0002):
        import subprocess
        self.max_mhz, self._proc, self._t0 = None, None, None
        try:
            self._proc = subprocess.Popen([sys.executable, "-c", self.CHILD, str(index), str(period_s)],
                                          stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            first = self._proc.stdout.readline().split()          # the child is up and sampling from here on
            self.max_mhz = int(first[1]) if len(first) == 2 and first[0] == "max" else None
        except Exception:
            self._proc = None

    def start(self):
        self._t0 = time.time()

    def mark(self):
        """End of a window that began at start(); returns its (t0, t1)."""
        return (self._t0, time.time())

    def stop(self, windows=None):
        """Ends the child; the summary covers start() .. now, plus a sample count per named window."""
        t1 = time.time()
        rows = []
        if self._proc:
            time.sleep(0.003)                                       # let the last samples through the pipe
            self._proc.terminate()
            try:
                out, _ = self._proc.communicate(timeout=5)
            except Exception:
                self._proc.kill()
                out = ""
            for line in out.splitlines():
                f = line.split()
                if len(f) == 3:
                    rows.append((float(f[0]), int(f[1]), int(f[2])))
        t0 = self._t0 if self._t0 is not None else 0.0
        inside = [r for r in rows if t0 <= r[0] <= t1]
        reasons = 0
        for r in inside:
            reasons |= r[2]
        res = {
            "sm_mhz": float(np.median([r[1] for r in inside])) if inside else None,
            "sm_max_mhz": self.max_mhz,
            "reasons": sorted(n for bit, n in self.REASONS.items() if reasons & bit),
            "samples": len(inside),
        }
        for name, (a, b) in (windows or {}).items():
            res["samples_in_" + name] = sum(1 for r in rows if a <= r[0] <= b)
        return res


# --------------------------------------------------------------------------- CPU oracle arm
def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def oracle_steps(w, n_steps: int, warmup: int = 0, budget_s: float = None, total_budget_s: float = None):
    """Run the CPU oracle (single-threaded byte loops, as it stands) over the workload's
    descriptor sets, one fence per step.  With ``total_budget_s`` every step is a bounded
    sample: the first ``m`` descriptors of its set, ``m`` chosen from one calibration step so
    that warmup + n_steps steps fit the budget.  Returns (seconds per step, bytes moved per
    step (read + written), descriptors per step)."""
    from oracle import Oracle
    imgs = [w.slot_image(s) for s in range(len(w.slot_sizes))]
    o = Oracle()
    for i in imgs:
        o.slot_register(i)
    frac = 1.0
    if total_budget_s is not None:
        t0 = time.perf_counter()
        assert o.memcpy_batch(w.epochs[0])[0] == 0 and o.fence() == 0
        t_full = time.perf_counter() - t0
        frac = min(1.0, total_budget_s / (t_full * (warmup + n_steps)))
    sets = [np.ascontiguousarray(e[: max(1, int(round(len(e) * frac)))]) for e in w.epochs]
    times, moved, units = [], [], []
    t_begin = time.perf_counter()
    for k in range(warmup + n_steps):
        e = sets[k % len(sets)]
        t0 = time.perf_counter()
        rc, _ = o.memcpy_batch(e)
        assert rc == 0
        assert o.fence() == 0
        dt = time.perf_counter() - t0
        if k >= warmup:
            times.append(dt)
            moved.append(2.0 * float(e["size"].sum()))
            units.append(len(e))
        if budget_s is not None and k >= warmup and time.perf_counter() - t_begin > budget_s:
            break
    return times, moved, units


def parallel_memcpy_baseline(w, budget_s: float):
    """The stronger CPU baseline of SURVEY.md S8(d): the same descriptor sets through libc memcpy,
    descriptors dealt to all host cores this process may use (oracle/parallel_memcpy.c; no
    validation, no counters -- a timing baseline, not the oracle)."""
    import oracle
    cores = host_cores()
    imgs = [w.slot_image(s) for s in range(len(w.slot_sizes))]
    sets = [np.ascontiguousarray(e) for e in w.epochs]
    oracle.parallel_memcpy_batch(imgs, sets[0], cores)            # warm-up (page faults, thread start)
    t_begin, times, moved = time.perf_counter(), [], []
    k = 0
    while time.perf_counter() - t_begin < budget_s:
        e = sets[k % len(sets)]
        t0 = time.perf_counter()
        oracle.parallel_memcpy_batch(imgs, e, cores)
        times.append(time.perf_counter() - t0)
        moved.append(2.0 * float(e["size"].sum()))
        k += 1
    return {"value": sum(moved) / sum(times) / 1e9, "unit": UNIT, "cores": cores, "kind": "libc memcpy per descriptor, all cores",
            "sample": "%d full steps of the same workload in %.1f s" % (len(times), sum(times))}


def size_decades(sizes):
    """Index arrays of the descriptors per size decade: [16, 160), [160, 1600), ...."""
    out, lo = [], 16
    sizes = np.asarray(sizes)
    while lo <= int(sizes.max()):
        idx = np.nonzero((sizes >= lo) & (sizes < 10 * lo))[0]
        if idx.size:
            out.append((lo, 10 * lo, idx))
        lo *= 10
    return out


def bytes_per_step(w) -> float:
    return 2.0 * w.bytes_copied / len(w.epochs)


def descs_per_step(w) -> float:
    return w.n_descs / len(w.epochs)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = make_workload(args.config)
    times, moved, units = oracle_steps(w, args.steps, warmup=args.warmup, total_budget_s=args.reference_seconds)
    total = float(sum(times))
    gbs = sum(moved) / total / 1e9
    full = descs_per_step(w)
    line = {
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": UNIT, "n_gpus": args.gpus,
        "steps": len(times), "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": WORKLOAD_TEXT[args.config], "name": args.config},
        "descs_per_s": sum(units) / total,
        "cpu_baseline": {"value": gbs, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": "%d steps, each the first %d of the %d descriptors of its set; "
                                   "host cores available: %d" % (len(times), units[0], full, host_cores())},
        "e2e": {"value": gbs, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------- CUDA arm
def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def pin_rate_gbs(device: int = 0):
    """Memory clock x 2 x bus width / 8 from the device properties (3996 MHz x 2 x 7680 bit / 8 =
    7672 GB/s on B200): the second denominator of SURVEY.md S8(d).  The measured peak is a
    torch copy calibration, not a ceiling: long streaming copies of this engine exceed it."""
    try:
        import torch
        p = torch.cuda.get_device_properties(device)
        return float(p.memory_clock_rate) * 1e3 * 2.0 * float(p.memory_bus_width) / 8.0 / 1e9
    except Exception:
        return None


def cross_gpu_leg(hicr, ctx, rank, world, group, stream, steps=20, pages=16384, page=4096, timeout_ms=30000):
    """N > 1 only: every rank volunteers a window as a Global Memory Slot
     and PUTS `pages` pages of `page` bytes per step into the window of rank + 1
    (Local-to-Global) with its own copy kernels over the peer mapping; a step ends in
    the initiator's blocking fence, the leg in one global fence whose count exchange must find
    every owner's totals.  Returns this rank's numbers; the control plane is `group` (gloo)."""
    import torch
    rng = np.random.default_rng(W.BASE_SEED + 7000 + rank)
    nbytes = pages * page
    src = torch.from_numpy(rng.integers(0, 256, nbytes, dtype=np.uint8)).cuda()
    win = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
    s_src, s_win = ctx.slot_register(src), ctx.slot_register(win)
    g = hicr.collective.exchange_global_slots(ctx, 77, [(rank, s_win)], group=group)
    peer = (rank + 1) % world
    d = W.make_descs([g[peer]] * pages, [s_src] * pages, rng.permutation(pages).astype(np.uint64) * page,
                     rng.permutation(pages).astype(np.uint64) * page, [page] * pages)
    t = torch.from_numpy(d.view(np.uint8).copy()).cuda()
    for _ in range(3):
        ctx.memcpy_batch(t, n=pages)
        ctx.fence()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        ctx.memcpy_batch(t, n=pages)
        ctx.fence()
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    t0 = time.perf_counter()
    hicr.collective.fence_global(ctx, group=group, timeout_ms=timeout_ms)
    gf_ms = 1e3 * (time.perf_counter() - t0)
    sent, recv = ctx.global_counters(s_win)
    # what landed in this rank's window is what rank - 1 put: same seeded source and page permutations
    prng = np.random.default_rng(W.BASE_SEED + 7000 + (rank - 1) % world)
    psrc = prng.integers(0, 256, nbytes, dtype=np.uint8).reshape(pages, page)
    dperm, sperm = prng.permutation(pages), prng.permutation(pages)
    expect = np.empty_like(psrc)
    expect[dperm] = psrc[sperm]
    ok = bool(torch.equal(win.cpu(), torch.from_numpy(expect.reshape(-1))))
    return {"put_ms_per_step": ms, "put_GBs": 2.0 * nbytes / (ms * 1e-3) / 1e9, "pages": pages, "page_bytes": page,
            "global_fence_ms": gf_ms, "owner_recv_total": int(recv), "owner_recv_expected": int((steps + 3) * pages),
            "window_equals_peer_source": ok, "peer": peer}


def other_configs_brief(hicr, torch, device, budget_s=20.0):
    """BASELINE.json's metric names more than config 2 ("descriptors/s + fence"): the full-size configs 1 and 4,
    each on a context and stream of its own, timed with CUDA events like `value`.  They ride in the default
    line as `other_configs` so that whoever runs bench.py records them too; the 16 GiB configs (3a, 3b) and the
    channel runs (5a, 5b) take too long to set up for that and keep their own --config runs."""
    out = {}
    t_all = time.perf_counter()
    for name, what in (("tiny", "device"), ("chain", "device"), ("chain_graph", "graph")):
        if time.perf_counter() - t_all > budget_s:
            out[name] = {"skipped": "time budget of the side measurements used up"}
            continue
        try:
            w = make_workload(name, 0)
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream):
                ctx = hicr.Context(device, stream.cuda_stream)
                try:
                    bufs = [torch.from_numpy(w.slot_image(s)).cuda() for s in range(len(w.slot_sizes))]
                    for b in bufs:
                        ctx.slot_register(b)
                    tabs = [torch.from_numpy(np.ascontiguousarray(e).view(np.uint8).copy()).cuda() for e in w.epochs]
                    ptrs, n_per, n_sets = [t.data_ptr() for t in tabs], [len(e) for e in w.epochs], len(w.epochs)
                    stream.synchronize()
                    graph = None
                    if what == "graph":
                        ctx.graph_begin(max(n_per))
                        for i in range(n_sets):
                            ctx.memcpy_batch(ptrs[i], n_per[i])
                            ctx.fence_async()
                        graph = ctx.graph_end()

                    def run(k):
                        if graph is None:
                            for i in range(k):
                                ctx.memcpy_batch(ptrs[i % n_sets], n_per[i % n_sets])
                                ctx.fence()
                        else:
                            for _ in range(k // n_sets):
                                graph.launch()
                                ctx.fence()

                    K = 10 * n_sets if n_sets > 1 else 2000          # config 4: ten passes over its 64 epochs
                    run(max(3, n_sets))
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    l0 = ctx.launch_count()
                    e0.record(stream)
                    run(K)
                    e1.record(stream)
                    torch.cuda.synchronize()
                    ms = e0.elapsed_time(e1) / K
                    out[name] = {"workload": WORKLOAD_TEXT[name], "steps": K, "us_per_step": 1e3 * ms,
                                 "value": bytes_per_step(w) / (ms * 1e-3) / 1e9, "unit": UNIT,
                                 "descs_per_s": descs_per_step(w) / (ms * 1e-3), "gpu_launches": int(ctx.launch_count() - l0),
                                 "step": "one epoch: one batch + one fence" + (" (stream-ordered inside the graph, one blocking "
                                         "fence per replay of 64)" if graph is not None else " (blocking)")}
                    if graph is not None:
                        graph.close()
                finally:
                    ctx.close()
        except Exception as exc:       # a side measurement must never cost the line
            out[name] = {"error": repr(exc)[:200]}
    return out


def run_cuda(args):
    import torch
    import paper_2509_01425_b200 as hicr

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback "
                         "(use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    w = make_workload(args.config, rank)
    stream = torch.cuda.Stream()
    n_sets = len(w.epochs)
    # at least 3 warm-up steps, and every rotating descriptor set once (the first use of a set is not a
    # steady-state step: cold TLB entries for its pages, the launch of a table not seen before)
    K, Wm = args.steps, max(3, args.warmup, n_sets if n_sets <= 8 else 3)
    with torch.cuda.stream(stream):
        ctx = hicr.Context(local, stream.cuda_stream)
        bufs = [torch.from_numpy(w.slot_image(s)).to("cuda", non_blocking=False) for s in range(len(w.slot_sizes))]
        ids = [ctx.slot_register(b) for b in bufs]
        host_tables = [np.ascontiguousarray(e) for e in w.epochs]
        dev_tables = [torch.from_numpy(t.view(np.uint8).copy()).cuda() for t in host_tables]
        n_per = [len(t) for t in host_tables]
        stream.synchronize()

        dev_ptrs = [t.data_ptr() for t in dev_tables]

        epoch_fence = ctx.fence_async if args.config == "chain_async" else ctx.fence

        def step_device(i):
            ctx.memcpy_batch(dev_ptrs[i % n_sets], n_per[i % n_sets])
            epoch_fence()

        def step_host(i):
            ctx.memcpy_batch(host_tables[i % n_sets])
            ctx.fence()

        graph = None
        if args.config == "chain_graph":
            # the 64 epochs recorded once; a replay = one hicr_graph_launch + one blocking fence
            ctx.graph_begin(max(n_per))
            for i in range(n_sets):
                ctx.memcpy_batch(dev_ptrs[i], n_per[i])
                ctx.fence_async()
            graph = ctx.graph_end()
            K = n_sets * max(1, -(-K // n_sets))      # whole replays only

        def run_steps(k):
            if graph is None:
                for i in range(k):
                    step_device(i)
            else:
                for _ in range(max(1, -(-k // n_sets))):
                    graph.launch()
                    ctx.fence()

        # ---- device-resident arm (value): K steps, nothing else on the stream
        clocks = ClockSampler(local)     # (its process is up and sampling before the warm-up is over)
        run_steps(Wm)
        ctx.fence()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        l0 = ctx.launch_count()
        clocks.start()
        t_host0 = time.perf_counter()
        e0.record(stream)
        run_steps(K)
        ctx.fence()                      # a no-op unless the epochs were closed by stream-ordered fences
        e1.record(stream)
        barrier()
        t_host = time.perf_counter() - t_host0
        clk_value_window = clocks.mark()            # the sampler keeps running over the other timed legs below
        launches = ctx.launch_count() - l0
        ms = e0.elapsed_time(e1)

        # ---- spread: every step of a second pass timed on its own with the host clock (a step ends in a
        # blocking fence, so the host sees its whole duration; CUDA events per step would add ~2 us each)
        # -- best, median and mean over R >= 20 repetitions -- and the same K steps on ONE
        # descriptor set (warm: part of the set stays in the 126 MB L2) beside the rotating (cold) ones
        per_step, warm = None, None
        if graph is None and args.config != "chain_async":
            R = max(20, min(K, 400))
            ts = np.empty(R)
            for i in range(R):
                t0 = time.perf_counter()
                step_device(i)
                ts[i] = time.perf_counter() - t0
            per_step = {"repetitions": R, "best_us": 1e6 * float(ts.min()), "median_us": 1e6 * float(np.median(ts)),
                        "mean_us": 1e6 * float(ts.mean()), "clock": "host, around memcpy_batch + blocking fence"}
            w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for _ in range(3):
                step_device(0)
            w0.record(stream)
            for _ in range(K):
                step_device(0)
            w1.record(stream)
            torch.cuda.synchronize()
            warm_ms = w0.elapsed_time(w1) / K
            warm = {"ms_per_step": warm_ms, "value": bytes_per_step(w) / (warm_ms * 1e-3) / 1e9, "unit": UNIT,
                    "what": "the same descriptor set every step"}

        # ---- roofline leg: the same K steps again with the library's CUDA events recorded
        # around every engine-kernel launch on the context's stream (they cost about 2 us per
        # step, which is why the `value` loop above runs without them)
        ctx.profile_enable(True)
        prof = np.zeros(4)
        for i in range(K):
            ctx.memcpy_batch(dev_ptrs[i % n_sets], n_per[i % n_sets])
            ctx.fence()
            prof += np.asarray(ctx.profile_read())
        n_prof = K
        ctx.profile_enable(False)

        # ---- config 3: GB/s per size decade -- the descriptors of each decade as a batch of their own
        per_decade = None
        if args.config in ("heavy_a", "heavy_b", "heavy_b_aligned"):
            per_decade = []
            for lo, hi, idx in size_decades(host_tables[0]["size"]):
                sub = np.ascontiguousarray(host_tables[0][idx])
                t = torch.from_numpy(sub.view(np.uint8).copy()).cuda()
                reps = 5
                for _ in range(2):
                    ctx.memcpy_batch(t, n=len(sub))
                    ctx.fence()
                d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                d0.record(stream)
                for _ in range(reps):
                    ctx.memcpy_batch(t, n=len(sub))
                    ctx.fence()
                d1.record(stream)
                torch.cuda.synchronize()
                dms = d0.elapsed_time(d1) / reps
                nb = 2.0 * float(sub["size"].sum())
                per_decade.append({"bytes_from": lo, "bytes_below": hi, "descs": int(len(sub)), "us": 1e3 * dms,
                                   "GBs": nb / (dms * 1e-3) / 1e9, "descs_per_s": len(sub) / (dms * 1e-3)})

        # ---- fence cost alone: an epoch with one 1-descriptor batch
        one = dev_tables[0]
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(3):
            ctx.memcpy_batch(one, n=1)
            ctx.fence()
        torch.cuda.synchronize()
        tf = time.perf_counter()
        for _ in range(50):
            ctx.memcpy_batch(one, n=1)
            ctx.fence()
        fence_us = (time.perf_counter() - tf) / 50 * 1e6

        # ---- end-to-end arm: host descriptor tables in, counters out, every step
        for i in range(Wm):
            step_host(i)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        g0.record(stream)
        for i in range(K):
            step_host(i)
        g1.record(stream)
        barrier()
        ms_e2e = g0.elapsed_time(g1)
        clk = clocks.stop({"value_leg": clk_value_window})
        clk["covers"] = "value, spread, warm, roofline and end-to-end legs (0.2 ms period, sampled by a separate process)"
        counters = [ctx.slot_counters(s) for s in ids]

        # ---- N > 1: the cross-GPU put of SURVEY.md S8(e) beside the per-rank number (never inside it)
        cross = None
        if world > 1:
            try:
                import datetime
                gloo = dist.new_group(backend="gloo", timeout=datetime.timedelta(seconds=120))
                ctx.instance_set(rank, world)
                mine = cross_gpu_leg(hicr, ctx, rank, world, gloo, stream)
                allr = [None] * world
                dist.all_gather_object(allr, mine, group=gloo)
                cross = {"what": "every rank puts 64 MiB per step into the Global Memory Slot of rank + 1 (4 KiB pages, "
                                 "random permutation), initiator's copy kernels over the CUDA-IPC peer mapping; "
                                 "unmeasured on hardware until a multi-GPU record exists",
                         "put_GBs_total": sum(r["put_GBs"] for r in allr), "put_ms_per_step_max": max(r["put_ms_per_step"] for r in allr),
                         "global_fence_ms_max": max(r["global_fence_ms"] for r in allr),
                         "counts_ok": all(r["owner_recv_total"] == r["owner_recv_expected"] for r in allr),
                         "data_ok": all(r["window_equals_peer_source"] for r in allr)}
            except Exception as exc:
                cross = {"error": repr(exc)[:300]}

    others = None
    if args.config == "bulk" and world == 1 and not args.no_other_configs:
        others = other_configs_brief(hicr, torch, local)

    ms_max, ms_e2e_max = rank_max(ms, dist, "cuda"), rank_max(ms_e2e, dist, "cuda")
    bps, dps = bytes_per_step(w), descs_per_step(w)
    agg = shard_report([bps * K] * world, [dps * K] * world, ms_max, K)
    agg_e2e = shard_report([bps * K] * world, [dps * K] * world, ms_e2e_max, K)

    if rank == 0:
        peak, peak_src = load_peaks()
        pin = pin_rate_gbs(local)
        prof /= max(1, n_prof)
        kernel_ms = {"plan_phase": prof[0], "copy_phase": prof[1], "engine_kernel_globaltimer": prof[2],
                     "engine_kernel": prof[3]}
        dom = "engine_kernel"          # the one kernel of a step; duration from CUDA events around its launch
        achieved = bps / (kernel_ms[dom] * 1e-3) / 1e9 if kernel_ms[dom] > 0 else 0.0
        traffic = None
        # dram__bytes_read.sum + dram__bytes_write.sum of that kernel per launch, from the
        # committed `ncu --set full` summary (profiles/traffic.csv), never measured here
        tp = os.path.join(ROOT, "profiles", "traffic.csv")
        if os.path.exists(tp):
            try:
                import csv
                for row in csv.DictReader(open(tp)):
                    if row["config"] == args.config and row["kernel"] == dom:
                        traffic = float(row["dram_bytes_read_per_launch"]) + float(row["dram_bytes_write_per_launch"])
            except Exception:
                traffic = None
        # CPU oracle beside it, same workload, bounded to about 10 s of CPU work
        cpu = None
        if not args.no_cpu_baseline:
            times, moved, _ = oracle_steps(make_workload(args.config, 0), 10 ** 6, warmup=1, budget_s=args.cpu_seconds)
            cpu_gbs = sum(moved) / float(sum(times)) / 1e9
            cpu = {"value": cpu_gbs, "unit": UNIT, "cores": 1, "kind": "oracle",
                   "sample": "%d full steps of the same workload in %.1f s (host cores available: %d)"
                             % (len(times), sum(times), host_cores())}
        cpu_par = None
        if not args.no_cpu_baseline:
            try:
                cpu_par = parallel_memcpy_baseline(make_workload(args.config, 0), args.cpu_seconds / 2)
            except Exception as exc:   # a baseline must never cost the line
                cpu_par = {"error": repr(exc)}
        line = {
            "metric": METRIC, "value": agg["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": agg["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8", "data": "synthetic",
            "config": {"workload": WORKLOAD_TEXT[args.config], "name": args.config,
                       "descriptor_tables": "device-resident", "l2": "inputs larger than L2: %d MiB touched per step, "
                       "%d rotating disjoint sets" % (bps / 2 ** 20, n_sets), "sharding": "independent slots per rank"},
            "descs_per_s": agg["descs_per_s"], "fence_us": fence_us, "host_ms_per_step": 1e3 * t_host / K,
            "per_step": per_step, "warm": warm, "per_size_decade": per_decade,
            "frac_of_hbm_peak": agg["value"] / world / peak,
            "e2e": {"value": agg_e2e["value"], "unit": UNIT,
                    "h2d_bytes_per_step": int(32 * dps), "d2h_bytes_per_step": int(64 + 16 * len(ids)),
                    "ms_per_step": agg_e2e["ms_per_step"], "what": "host descriptor tables in, slot counters out"},
            "gpu_launches": int(launches),
            "kernel_ms": kernel_ms,
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": UNIT,
                         "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                         # the same kernel time against the DRAM bytes ncu counted (writes still dirty in L2 at
                         # kernel end are paid for by the next step): the fraction by bytes actually moved
                         "frac_by_dram_traffic": (traffic / (kernel_ms[dom] * 1e-3) / 1e9 / peak) if traffic and kernel_ms[dom] > 0 else None,
                         "algorithmic_bytes_per_launch": bps, "pin_rate": pin,
                         "frac_of_pin_rate": (achieved / pin) if pin else None},
            "cross_gpu": cross,
            "other_configs": others,
            "cpu_baseline": cpu, "cpu_baseline_parallel": cpu_par,
            "clocks": clk,
            "counters_ok": bool(sum(c[0] for c in counters) == sum(c[1] for c in counters)),
        }
        print(json.dumps(line))
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


# --------------------------------------------------------------------------- channel configs
CHANNEL_TEXT = {
    "spsc_stream": "config 5a SPSC, device-resident run: 256 B tokens, capacity 1024, 2^24 tokens, batches U{1..1024}, "
                   "one kernel: a thread-block cluster with two producer CTAs and two consumer CTAs on the one ring",
    "spsc_calls": "config 5a SPSC, host-call path: push(b_i) then pop(max = capacity), one launch per call",
    "mpsc": "config 5b non-locking MPSC: 148 producers (one CTA per SM), 64 B tokens, 2^20 tokens each, rings of 1024, "
            "one logical consumer = one consumer CTA per ring (producer and consumer of a ring form a thread-block cluster)",
    "mpsc_locking": "config 5b's shape in the paper's LOCKING mode (SURVEY.md S8(f) 2): 148 producers share ONE ring of 1024 "
                    "tokens of 64 B through atomic reservation and in-order commit, 2^20 tokens each, single consumer CTA",
}


def run_pingpong(args):
    """the paper's Test Case 1 on the built channel --
    two opposing SPSC channels of capacity 1 between two endpoints, message sizes log-spaced
    from 1 B to 2^31 B, 10 repetitions each with standard deviation, goodput G(s) = 2 s / RTT.
    One round trip = push(A->B), pop at B, push(B->A), pop at A through the host-call API
    (every call complete on return).  Shape only: the paper's curve is two hosts over
    InfiniBand; here both endpoints are buffers in one B200's HBM."""
    import torch
    import paper_2509_01425_b200 as hicr
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(0)
    reps, warm = 10, 2
    sizes = [4 ** k for k in range(0, 16)] + [1 << 31]
    stream = torch.cuda.Stream()
    sweep = []
    clocks = ClockSampler(0)
    clocks.start()
    launches = 0
    ok = True
    with torch.cuda.stream(stream):
        ctx = hicr.Context(0, stream.cuda_stream)
        smax = max(sizes)
        rng = np.random.default_rng(W.BASE_SEED + 6)
        store = [torch.zeros(smax, dtype=torch.uint8, device="cuda") for _ in range(4)]   # ring AB, ring BA, buf A, buf B
        store[2][: 1 << 20] = torch.from_numpy(rng.integers(0, 256, 1 << 20, dtype=np.uint8)).cuda()
        for s in sizes:
            view = [t[:s] for t in store]
            ids = [ctx.slot_register(v) for v in view]
            ab, ba = ctx.channel_create(ids[0], s, 1), ctx.channel_create(ids[1], s, 1)
            view[3].zero_()
            stream.synchronize()
            l0 = ctx.launch_count()
            rtt = []
            for r in range(warm + reps):
                t0 = time.perf_counter()
                assert ab.push(ids[2], 0, 1) == 1
                assert ab.pop(ids[3], 0, 1) == 1
                assert ba.push(ids[3], 0, 1) == 1
                assert ba.pop(ids[2], 0, 1) == 1
                dt = time.perf_counter() - t0
                if r >= warm:
                    rtt.append(dt)
            launches += ctx.launch_count() - l0
            ok = ok and bool(torch.equal(view[2], view[3])) and ab.counters() == (warm + reps, warm + reps)
            ab.close()
            ba.close()
            for i in ids:
                ctx.slot_unregister(i)
            m, sd = float(np.mean(rtt)), float(np.std(rtt))
            sweep.append({"bytes": s, "rtt_us": 1e6 * m, "rtt_us_std": 1e6 * sd, "goodput_GBs": 2.0 * s / m / 1e9})
        ctx.close()
    clk = clocks.stop()
    peak, peak_src = load_peaks()
    big = sweep[-1]
    line = {
        "metric": "ping-pong goodput 2 s / RTT over two opposing capacity-1 channels", "value": big["goodput_GBs"],
        "unit": UNIT, "n_gpus": 1, "steps": reps, "warmup": warm, "ms_per_step": big["rtt_us"] / 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": "paper Test Case 1 shape: message sizes 1 B .. 2^31 B, 10 repetitions each; value = largest size",
                   "name": "pingpong", "l2": "largest sizes exceed L2; small sizes are latency-bound by construction"},
        "sweep": sweep, "gpu_launches": int(launches),
        "e2e": {"value": big["goodput_GBs"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 4 * 40,
                "what": "host wall clock around four blocking calls per round trip"},
        # one round trip moves s bytes four times (read + write each): 8 s of HBM traffic
        "roofline": {"bound": "hbm", "kernel": "channel_call_kernel", "achieved": 8.0 * big["bytes"] / (big["rtt_us"] * 1e-6) / 1e9,
                     "peak": peak, "unit": UNIT, "frac": 8.0 * big["bytes"] / (big["rtt_us"] * 1e-6) / 1e9 / peak,
                     "traffic": None, "peak_source": peak_src},
        "cpu_baseline": None, "clocks": clk, "echo_equals_message": bool(ok),
    }
    print(json.dumps(line))
    return 0


def oracle_channel_sample(w, budget_s: float):
    """cpu_baseline of the channel configs: the oracle's push / pop(max = C) loop, token by token,
    on ONE ring (producer 0's batches and source prefix), until ``budget_s`` of CPU time."""
    from oracle import Oracle
    T, C = w.token_bytes, w.capacity
    batches = w.batches[0]
    n_cap = int(min(w.n_tokens, 1 << 22))                       # at most 2^22 tokens of the source prefix
    src = np.random.default_rng(w.seed).integers(0, 256, n_cap * T, dtype=np.uint8)   # timing only: any bytes do
    ring, sink = np.zeros(T * C, np.uint8), np.zeros(n_cap * T, np.uint8)
    o = Oracle()
    r, s, k = o.slot_register(ring), o.slot_register(src), o.slot_register(sink)
    _, ch = o.channel_create(r, T, C)
    pos, nb = 0, 0
    t0 = time.perf_counter()
    for b in batches:
        b = int(b)
        if pos + b > n_cap or time.perf_counter() - t0 > budget_s:
            break
        o.channel_push(ch, s, pos * T, b)
        o.channel_pop(ch, k, pos * T, C)
        pos += b
        nb += 1
    dt = time.perf_counter() - t0
    return {"value": 4.0 * pos * T / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle", "tokens_per_s": pos / dt,
            "sample": "push / pop(max = C) of the first %d batches (%d tokens of %d B) of one ring in %.1f s "
                      "(host cores available: %d)" % (nb, pos, T, dt, host_cores())}


def run_channel(args):
    """Configs 5a / 5b.  A step is the whole push/pop sequence; bytes = 4 x payload (source ->
    ring -> sink, read + write each hop).  value = device time of the sequence; e2e = the
    same through the host-call API where there is one (spsc_calls), else the same number
    with the host wall clock around the blocking call."""
    import torch
    import paper_2509_01425_b200 as hicr
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(0)
    K, Wm = args.steps, max(1, args.warmup)
    name = args.config
    if name in ("mpsc", "mpsc_locking"):
        w = W.mpsc() if args.tokens is None else W.mpsc(n_tokens=args.tokens)
    else:
        w = W.spsc() if args.tokens is None else W.spsc(n_tokens=args.tokens)
    T, C, P, N = w.token_bytes, w.capacity, w.producers, w.n_tokens
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = hicr.Context(0, stream.cuda_stream)
        locking = name == "mpsc_locking"
        rings = [torch.zeros(T * C, dtype=torch.uint8, device="cuda") for _ in range(1 if locking else P)]
        if locking:
            srcs = [torch.from_numpy(a).cuda() for a in W.generators.tagged_sources(P, N, T)]
            sinks = [torch.zeros(P * N * T, dtype=torch.uint8, device="cuda")]
        else:
            srcs = [torch.from_numpy(w.source_image(p)).cuda() for p in range(P)]
            sinks = [torch.zeros(N * T, dtype=torch.uint8, device="cuda") for _ in range(P)]
        rid = [ctx.slot_register(t) for t in rings]
        sid = [ctx.slot_register(t) for t in srcs]
        kid = [ctx.slot_register(t) for t in sinks]
        stream.synchronize()
        if locking:
            ch = ctx.channel_create(rid[0], T, C)
            def step():
                ch.locking_stream(sid, kid[0], 0, N, 256)
        elif name == "mpsc":
            m = ctx.mpsc_create(rid, T, C)
            def step():
                m.stream(sid, kid, N, 256)
        else:
            ch = ctx.channel_create(rid[0], T, C)
            batches = w.batches[0]
            if name == "spsc_stream":
                def step():
                    ch.stream(sid[0], 0, kid[0], 0, batches)
            else:
                def step():
                    pos = 0
                    for b in batches:
                        b = int(b)
                        k = ch.push(sid[0], pos * T, b)
                        k2 = ch.pop(kid[0], pos * T, C)
                        assert k == b == k2
                        pos += b
        for _ in range(Wm):
            step()
        clocks = ClockSampler(0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        l0 = ctx.launch_count()
        clocks.start()
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(K):
            step()
        e1.record(stream)
        torch.cuda.synchronize()
        t_host = time.perf_counter() - t0
        clk = clocks.stop()
        launches = ctx.launch_count() - l0
        ms = e0.elapsed_time(e1)
        if locking:
            # the interleaving is not defined: per-producer FIFO and "every token once", from the tags
            tags = sinks[0].view(torch.int32).view(P * N, T // 4)[:, :2]
            order = torch.sort(tags[:, 0].to(torch.int64), stable=True).indices
            key = tags[order, 0].to(torch.int64) * N + tags[order, 1].to(torch.int64)
            ok = bool(torch.equal(key, torch.arange(P * N, device="cuda")))
            del key, tags
            allsrc = torch.cat(srcs).view(P * N, T)
            ok = ok and bool(torch.equal(sinks[0].view(P * N, T)[order], allsrc))
            del allsrc, order
        else:
            ok = all(torch.equal(a, b) for a, b in zip(srcs, sinks))
    tokens = float(P) * N
    bytes_step = 4.0 * tokens * T
    peak, peak_src = load_peaks()
    gbs = bytes_step * K / (ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": gbs, "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": Wm, "ms_per_step": ms / K,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": CHANNEL_TEXT[name], "name": name, "tokens": int(tokens), "token_bytes": T,
                   "l2": "inputs larger than L2: %d MiB of source and sink per step" % (2 * tokens * T / 2 ** 20)},
        "tokens_per_s": tokens * K / (ms * 1e-3),
        "e2e": {"value": bytes_step * K / t_host / 1e9, "unit": UNIT,
                "h2d_bytes_per_step": int(8 * len(w.batches[0])) if name == "spsc_stream" else 0,
                "d2h_bytes_per_step": 32 * (2 * len(w.batches[0]) if name == "spsc_calls" else 1),
                "ms_per_step": 1e3 * t_host / K, "what": "host wall clock around the blocking calls"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "kernel": {"mpsc": "pipe_cluster_kernel", "spsc_stream": "pipe_cluster_kernel", "mpsc_locking": "mpsc_locking_kernel"}.get(name, "channel_call_kernel"),
                     "achieved": gbs / 2, "peak": peak, "unit": UNIT, "frac": gbs / 2 / peak, "traffic": None,
                     "peak_source": peak_src,
                     "note": "DRAM sees source and sink only (the ring lives in L2): algorithmic DRAM bytes = 2 x payload; "
                             "what binds is the lap of a ring (write -> publish -> read -> publish), see profiles/r02_channels.md"},
        "cpu_baseline": None if args.no_cpu_baseline else oracle_channel_sample(w, args.cpu_seconds),
        "clocks": clk, "sink_equals_source": bool(ok),
    }
    print(json.dumps(line))
    ctx.close()
    return 0


def spawn_command(n_gpus, argv, port=None):
    """The launch line of the contract: one rank per GPU of this node, rendezvous on 127.0.0.1."""
    if port is None:
        import socket
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n_gpus),
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def main(argv=None):
    argv = list(sys.argv[1:] if argv is None else argv)
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", default="bulk", choices=sorted(WORKLOAD_TEXT) + sorted(CHANNEL_TEXT) + ["pingpong"])
    ap.add_argument("--tokens", type=int, default=None, help="channel configs: tokens per producer (default: full size)")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="default run: leave out the side measurements of configs 1 and 4 (`other_configs`)")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="CPU work of the cpu_baseline leg")
    ap.add_argument("--reference-seconds", type=float, default=90.0,
                    help="--impl reference: CPU work of the whole run (each step a bounded sample)")
    args = ap.parse_args(argv)
    if args.config == "pingpong":
        return run_pingpong(args)
    if args.config in CHANNEL_TEXT:
        if args.impl == "reference":
            raise SystemExit("--impl reference times the memcpy configs only")
        args.steps = min(args.steps, 3) if args.steps == 2000 else args.steps
        return run_channel(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` without a launcher: start the N ranks ourselves (the same line the
        # driver uses); rank 0 of them prints the JSON line
        import subprocess
        import torch
        if torch.cuda.device_count() < args.gpus:
            raise SystemExit("bench.py: --gpus %d but this node has %d CUDA device(s)" % (args.gpus, torch.cuda.device_count()))
        return subprocess.call(spawn_command(args.gpus, argv))
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
