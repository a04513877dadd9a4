// hicr_copy.cu -- hicr_memcpy_batch: descriptor ingest + validation (a2), binning and
// work expansion (a3), the copies (a4, a5) and counter accumulation (a6), as ONE
// persistent cooperative kernel per batch.
//
// The operation: the Communication Manager's memcpy, "specify the source and
// destination memory slots, as well as the offsets within them and the size of data to
// communicate ... the operation will be initiated. Otherwise, it will be rejected"
// (PAPER.md:373), batched; completion deferred to the fence.
//
// engine_kernel, grid = SMs x kCtasPerSm co-resident CTAs of 256 threads:
//   phase A  one thread per descriptor (grid-stride tiles): validate against the slot
//            table, resolve absolute addresses, expand descriptors above 8 KiB into the chunk
//            queue (warp ballot + warp prefix sum + one atomic per warp), count messages per
//            slot in a shared-memory histogram; small descriptors stay in the table.
//   barrier  grid-wide, ONE 64-bit word: arrivals, "saw an invalid descriptor" votes, "my small
//            descriptors are team-sized" votes and the chunk-queue length share it, so the
//            poll that sees the last arrival also delivers the verdict.  Any invalid
//            descriptor: nothing is copied or counted (all-or-nothing).  While the barrier
//            fills, every warp prefetches the sources of its first descriptors into L2.
//            Host-validated tables without large descriptors skip the barrier.
//   phase B  histogram flushed into the cumulative u64 counters (one atomic per touched
//            slot per CTA).  B1, CTA per 128 KiB chunk: dynamic tickets, thread 0 two rounds
//            ahead (next item loaded, ticket after that in flight); 16 B-aligned chunks go
//            through 1-D TMA bulk copies staged in shared memory, the rest through 16 B vector
//            loads / aligned stores with byte-shifted sources (copy_span).  B2, small
//            descriptors read from the table in place: warp tickets by guided self-scheduling
//            (three in flight per warp), or equal static shares when the batch is team-sized;
//            > 256 B: copy_span by the warp; <= 256 B: copy_team, eight descriptors at a time
//            by teams of four lanes, every load before the first store.
//   finish   the last CTA to finish pushes the counters and the completion record into
//            mapped pinned host memory (what hicr_fence polls) and clears the control block.
#include "hicr_internal.cuh"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

namespace hicr {

__device__ __forceinline__ void report_bad(Ctl *ctl, uint64_t index, unsigned id)
{
    atomicMax(&ctl->bad_inv, ~((unsigned long long)index << 4 | id));
}

__device__ __forceinline__ unsigned long long globaltimer()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void put_item(WorkItem *q, uint64_t src, uint64_t dst, uint64_t size)
{
    uint4 *p = reinterpret_cast<uint4 *>(q);
    p[0] = make_uint4((unsigned)src, (unsigned)(src >> 32), (unsigned)dst, (unsigned)(dst >> 32));
    p[1] = make_uint4((unsigned)size, (unsigned)(size >> 32), 0, 0);
}

__device__ __forceinline__ WorkItem load_item(const WorkItem *q)
{
    const uint4 *p = reinterpret_cast<const uint4 *>(q);
    const uint4 a = __ldcg(p), b = __ldcg(p + 1);
    WorkItem w;
    w.src = (uint64_t)a.x | ((uint64_t)a.y << 32);
    w.dst = (uint64_t)a.z | ((uint64_t)a.w << 32);
    w.size = (uint64_t)b.x | ((uint64_t)b.y << 32);
    w.pad = 0;
    return w;
}

// Chunks of a large descriptor.  From kAlignedSplitMin bytes on, the cuts sit at multiples of
// kChunkBytes of the DESTINATION address, so every chunk but the first starts 16 B-aligned
// (no byte head, and TMA-eligible when the source is congruent); below that, every
// kChunkBytes from the start.
constexpr uint64_t kAlignedSplitMin = 4 * kChunkBytes;
__device__ __forceinline__ unsigned chunk_count(uint64_t dst, uint64_t size)
{
    if (size >= kAlignedSplitMin) return (unsigned)((dst + size - 1) / kChunkBytes - dst / kChunkBytes + 1);
    return (unsigned)((size + kChunkBytes - 1) / kChunkBytes);
}
__device__ __forceinline__ void chunk_range(uint64_t dst, uint64_t size, unsigned c, uint64_t &off, uint64_t &len)
{
    if (size >= kAlignedSplitMin) {
        const uint64_t first = dst / kChunkBytes;
        const uint64_t lo = c == 0 ? dst : (first + c) * kChunkBytes;
        const uint64_t hi = min(dst + size, (first + c + 1) * kChunkBytes);
        off = lo - dst;
        len = hi - lo;
    } else {
        off = (uint64_t)c * kChunkBytes;
        len = min(kChunkBytes, size - off);
    }
}

struct EngineArgs {
    const hicr_desc_t *descs;
    uint64_t n;
    const SlotRow *slots;
    uint32_t n_slots;
    uint32_t tma_min;
    Ctl *ctl;
    WorkItem *chunk_q;
    uint64_t chunk_cap;
    SlotCnt *cnt;                    // [HICR_MAX_SLOTS] cumulative message counters
    HostRecord *rec_ring;            // kRecRing completion records (device alias of mapped pinned memory); batch number
                                     // seq (1-based, counted on the device in Ctl::seq) writes record (seq - 1) % kRecRing
                                     // with flag rec_flag(seq): nothing in the arguments names the launch, so a
                                     // captured launch can be replayed (hicr_graph_*)
    unsigned long long *push;        // [kPushWordsPerSlot * kPushSlots] pushed counter words (mapped pinned memory)
    uint32_t n_push;
    uint32_t skip_barrier;           // the host validated the table and it holds no large descriptor
    uint32_t hand_out;               // kHandOutVote (device tables), or what the host's own count says
    // Global Memory Slots: per table row of kind GLOBAL the address of the owner's
    // counters (peer-mapped when the owner is another instance), and this batch's counts per such row
    const uint64_t *gptr;
    SlotCnt *gdelta;
    uint32_t any_global;
};
constexpr uint32_t kHandOutVote = 0, kHandOutDynamic = 1, kHandOutStatic = 2;

// One 8-byte word of the completion record: payload in the low half, flag in the high half.
__device__ __forceinline__ void put_word(unsigned long long *w, uint32_t payload, uint32_t flag)
{
    *reinterpret_cast<volatile unsigned long long *>(w) = ((unsigned long long)flag << 32) | payload;
}

// Slot row `s` (s < n_slots): from the shared-memory cache when the table fits, else from L2.
__device__ __forceinline__ SlotRow slot_row(const SlotRow *cache, const SlotRow *global, uint32_t n_slots, uint32_t s)
{
    if (n_slots <= kSlotCache) return cache[s];
    const uint4 v = __ldg(reinterpret_cast<const uint4 *>(global + s));
    SlotRow r;
    r.base = (uint64_t)v.x | ((uint64_t)v.y << 32);
    r.meta = (uint64_t)v.z | ((uint64_t)v.w << 32);
    return r;
}

// The 32 bytes of one descriptor, issued now and consumed later (volatile: the loads stay
// where they are written, ahead of the copy they overlap with).
__device__ __forceinline__ void load_desc_raw(const hicr_desc_t *d, uint4 &lo, uint4 &hi)
{
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(lo.x), "=r"(lo.y), "=r"(lo.z), "=r"(lo.w) : "l"(d));
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(hi.x), "=r"(hi.y), "=r"(hi.z), "=r"(hi.w)
                 : "l"(reinterpret_cast<const unsigned char *>(d) + 16));
}

// Check one descriptor (its 32 bytes in lo, hi) against the slot table with THE validator
// (check_transfer, hicr_internal.cuh).  Returns 0 or the error id; on success src/dst are
// absolute addresses and ds/ss the table indices of the two slots.
__device__ __forceinline__ unsigned resolve(const uint4 &lo, const uint4 &hi, const SlotRow *cache,
                                            const SlotRow *global, uint32_t n_slots, uint32_t &ds, uint32_t &ss,
                                            uint64_t &dst, uint64_t &src, uint64_t &size)
{
    ds = lo.x & kSlotIndexMask;
    ss = lo.y & kSlotIndexMask;
    const uint64_t dst_off = (uint64_t)lo.z | ((uint64_t)lo.w << 32);
    const uint64_t src_off = (uint64_t)hi.x | ((uint64_t)hi.y << 32);
    size = (uint64_t)hi.z | ((uint64_t)hi.w << 32);
    SlotRow dr{0, kInvalidMeta}, sr{0, kInvalidMeta};
    const bool d_in = ds < n_slots, s_in = ss < n_slots;
    if (d_in) dr = slot_row(cache, global, n_slots, ds);
    if (s_in) sr = slot_row(cache, global, n_slots, ss);
    const unsigned bad = check_transfer(dr, d_in, lo.x, dst_off, sr, s_in, lo.y, src_off, size);
    if (bad) return bad;
    dst = dr.base + dst_off;
    src = sr.base + src_off;
    return 0;
}

// A descriptor of a batch already known to be valid: absolute addresses, and its size if it
// belongs to the warp-per-descriptor class (0 < size <= kSmallMax), else 0.
__device__ __forceinline__ unsigned resolve_small(const uint4 &lo, const uint4 &hi, const SlotRow *cache,
                                                  const SlotRow *global, uint32_t n_slots, uint64_t &dst, uint64_t &src)
{
    const uint64_t size = (uint64_t)hi.z | ((uint64_t)hi.w << 32);
    if (size == 0 || size > kSmallMax) return 0;
    dst = slot_row(cache, global, n_slots, lo.x & kSlotIndexMask).base + ((uint64_t)lo.z | ((uint64_t)lo.w << 32));
    src = slot_row(cache, global, n_slots, lo.y & kSlotIndexMask).base + ((uint64_t)hi.x | ((uint64_t)hi.y << 32));
    return (unsigned)size;
}

// One 128-byte line of a source range on its way into L2 (no register, no completion to
// wait for); only lines that hold a byte of the range are touched.
__device__ __forceinline__ void prefetch_l2_line(uint64_t addr)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(addr) : "memory");
}

// Shared-memory layout of the engine kernel (dynamic): TMA stages, slot cache, histogram.
constexpr size_t kSmemStages = (size_t)kWarps * kTmaStages * kTmaPiece;
constexpr size_t kSmemCache = (size_t)kSlotCache * sizeof(SlotRow);

__global__ void __launch_bounds__(kThreads, kCtasPerSm) engine_kernel(const EngineArgs a)
{
    extern __shared__ __align__(128) unsigned char dyn_smem[];   // [stages][slot cache][histogram]
    __shared__ uint64_t bars[kWarps * kTmaStages];
    __shared__ unsigned sh_ticket[2];
    __shared__ WorkItem sh_item[2];              // queue items of the current and the next chunk
    __shared__ unsigned sh_flag;
    __shared__ unsigned long long sh_seq;        // last CTA: this batch's sequence number
    __shared__ unsigned long long sh_sync;       // the barrier word as the last poll saw it
    __shared__ unsigned sh_first1;               // first descriptor of the CTA's second tickets (warp w: + w x cnt1)
    __shared__ unsigned sh_small[2];             // bytes and count of the small descriptors this CTA validated
    __shared__ unsigned char sh_rank[kWarps][32];   // per warp: lane of the r-th team-sized descriptor of the ticket
    SlotRow *cache = reinterpret_cast<SlotRow *>(dyn_smem + kSmemStages);
    unsigned int *hist = reinterpret_cast<unsigned int *>(dyn_smem + kSmemStages + kSmemCache);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    Ctl *ctl = a.ctl;
    const uint32_t n_slots = a.n_slots;
    const bool use_hist = n_slots <= kSmemSlotHist;
    if (blockIdx.x == 0 && tid == 0) ctl->t_start = globaltimer();
    // the first tile's descriptors are requested before anything else, so that their DRAM
    // round trip overlaps the slot-table fetch and the shared-memory set-up
    uint4 alo = make_uint4(0, 0, 0, 0), ahi = alo;
    const uint64_t tile0 = (uint64_t)blockIdx.x * kThreads;
    // A table the host has validated and that holds no large descriptor needs no pass of its own over the
    // descriptors: nothing to check, nothing to bin, and the messages are counted by the warp that copies
    // them (phase B2) -- so the copies start with the kernel, and a table that is read in place from pinned
    // host memory is fetched ticket by ticket behind them instead of once up front over PCIe.
    const bool lazy = a.skip_barrier && use_hist;
    if (!lazy && tile0 + tid < a.n) load_desc_raw(a.descs + tile0 + tid, alo, ahi);
    // ---- warp tickets of phase B2.  The first ticket of every warp is static (warp g owns
    // descriptors [g c0, (g+1) c0)); the others are atomics on a shared cursor that counts
    // from the end of the static tickets.
    const unsigned n = (unsigned)a.n, nw = gridDim.x * kWarps;
    const unsigned gdiv = kGss * nw;
    auto ticket_size = [&](unsigned total, unsigned seen) { return min(max((total - min(seen, total)) / gdiv, 1u), kMaxGroup); };
    // (a multiple of 8 when it can be: team-sized descriptors are copied 8 at a time)
    const unsigned cnt_static0 = ticket_size(n, 0), cnt_static = cnt_static0 >= 8 ? cnt_static0 & ~7u : cnt_static0;
    const unsigned static_end = nw * cnt_static;
    // ... and so are the descriptors of this warp's static first ticket: their round trip (cold: another
    // CTA's tile) hides behind phase A instead of sitting between it and the arrival at the barrier
    // ... and so is the CTA's ticket for its warps' second tickets: an index range only, and an L2 round
    // trip the arrival at the barrier would otherwise wait for (a release waits for the thread's own atomic)
    unsigned cnt1 = a.hand_out != kHandOutStatic ? ticket_size(n, static_end) : 0u, base1 = 0;
    if (tid == 0 && a.hand_out != kHandOutStatic) base1 = atomicAdd(&ctl->next_desc, cnt1 * kWarps);
    const unsigned first0_early = (blockIdx.x * kWarps + warp) * cnt_static;
    uint4 flo = make_uint4(0, 0, 0, 0), fhi = flo;
    const bool fhave = (unsigned)lane < cnt_static && first0_early + lane < n;
    if (fhave) load_desc_raw(a.descs + first0_early + lane, flo, fhi);
    if (n_slots <= kSlotCache)
        for (uint32_t i = tid; i < n_slots; i += kThreads) {
            const uint4 v = __ldg(reinterpret_cast<const uint4 *>(a.slots + i));
            cache[i].base = (uint64_t)v.x | ((uint64_t)v.y << 32);
            cache[i].meta = (uint64_t)v.z | ((uint64_t)v.w << 32);
        }
    if (use_hist)
        for (uint32_t i = tid; i < 2 * n_slots; i += kThreads) hist[i] = 0;
    if (tid < 2) sh_small[tid] = 0;
    TmaLane tma;
    tma.stage = dyn_smem + (size_t)warp * kTmaStages * kTmaPiece;
    tma.bar = &bars[warp * kTmaStages];
    tma.k = 0;
    tma.pend_dst = nullptr;
    tma.pend_len = 0;
    tma.stores = false;
    if (lane == 0) {
        for (int s = 0; s < kTmaStages; s++) mbar_init(tma.bar + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

    __syncthreads();

    // ================================================================ phase A (a2, a3, a6)
    bool bad_seen = false, wrote_chunks = false;
    unsigned small_bytes = 0, small_cnt = 0;
    for (uint64_t tile = lazy ? a.n : tile0; tile < a.n; tile += (uint64_t)gridDim.x * kThreads) {
        const uint64_t i = tile + tid;
        uint64_t src = 0, dst = 0, size = 0;
        uint32_t ss = 0, ds = 0;
        bool valid = false;
        if (i < a.n) {
            if (tile != tile0) load_desc_raw(a.descs + i, alo, ahi);
            const unsigned bad = resolve(alo, ahi, cache, a.slots, n_slots, ds, ss, dst, src, size);
            if (bad) {
                report_bad(ctl, i, bad);
                bad_seen = true;
            } else valid = true;
        }
        if (valid && size != 0 && size <= kSmallMax) {
            small_bytes += ((unsigned)size + 15u) >> 4;   // in 16 B units: a CTA's sum stays below 2^32
            small_cnt++;
        }

        // ---- (a6) one message per descriptor: sent on the source slot, recv on the destination
        // (lanes with the same slot elect one leader; invalid lanes carry a key no slot has)
        if (use_hist) {
            const unsigned ms = __match_any_sync(0xffffffffu, valid ? ss : 0xffffffffu);
            if (valid && lane == __ffs(ms) - 1) atomicAdd(&hist[ss], __popc(ms));
            const unsigned md = __match_any_sync(0xffffffffu, valid ? ds : 0xffffffffu);
            if (valid && lane == __ffs(md) - 1) atomicAdd(&hist[n_slots + ds], __popc(md));
        }

        // ---- (a3) binning.  Small descriptors (0 < size <= kSmallMax) stay in the table and are
        // copied from it in place; large ones are expanded into the chunk queue: warp ballot,
        // warp prefix sum of the chunk counts, one atomic per warp.
        const bool is_large = valid && size > kSmallMax;
        const unsigned large_mask = __ballot_sync(0xffffffffu, is_large);
        if (large_mask) {
            wrote_chunks = true;
            const unsigned nch = is_large ? chunk_count(dst, size) : 0u;
            unsigned incl = nch;   // inclusive warp scan of the chunk counts
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned v = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += v;
            }
            const unsigned total = __shfl_sync(0xffffffffu, incl, 31);
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(&ctl->sync, (unsigned long long)total << kSyncChunkShift) >> kSyncChunkShift;
            base = __shfl_sync(0xffffffffu, base, 0);
            const uint64_t my_first = base + (incl - nch);
            if (is_large && my_first + nch > a.chunk_cap) {
                report_bad(ctl, i, kBadNoCapacity);
                bad_seen = true;
            }
            // work expansion: the whole warp writes the chunk items of each large descriptor
            unsigned m = large_mask;
            while (m) {
                const int l = __ffs(m) - 1;
                m &= m - 1;
                const uint64_t s0 = __shfl_sync(0xffffffffu, src, l);
                const uint64_t d0 = __shfl_sync(0xffffffffu, dst, l);
                const uint64_t sz = __shfl_sync(0xffffffffu, size, l);
                const uint64_t first = __shfl_sync(0xffffffffu, my_first, l);
                const unsigned cnt = __shfl_sync(0xffffffffu, nch, l);
                if (first + cnt > a.chunk_cap) continue;
                for (unsigned c = lane; c < cnt; c += 32) {
                    uint64_t off, len;
                    chunk_range(d0, sz, c, off, len);
                    put_item(a.chunk_q + first + c, s0 + off, d0 + off, len);
                }
            }
        }
    }
    // this CTA's vote on how phase B2 hands out work: are its small descriptors team-sized on average?
#pragma unroll
    for (int d = 16; d; d >>= 1) {
        small_bytes += __shfl_xor_sync(0xffffffffu, small_bytes, d);
        small_cnt += __shfl_xor_sync(0xffffffffu, small_cnt, d);
    }
    if (lane == 0 && small_cnt) {
        atomicAdd(&sh_small[0], small_bytes);
        atomicAdd(&sh_small[1], small_cnt);
    }

    // the second ticket of every warp and the descriptors of the first are requested before
    // the barrier so that their latencies hide behind it.  Tickets are index ranges only;
    // nothing is written before the batch is known to be valid.
    // (ONE atomic per CTA for its eight warps' second tickets: 2368 same-address atomics at once
    // take microseconds to drain, and the CTA's arrival at the barrier waits for its own)
    unsigned first0 = (blockIdx.x * kWarps + warp) * cnt_static, first1 = 0;

    // ================================================================ grid barrier
    uint64_t src = 0, dst = 0;
    unsigned sz32 = 0;
    // (a6, lazy tables) one message per descriptor of a ticket, counted by the warp that holds it: the lanes
    // with the same slot elect one leader, which adds their number to the shared-memory histogram
    auto count_ticket = [&](bool have, const uint4 &lo) {
        const uint32_t ds_ = lo.x & kSlotIndexMask, ss_ = lo.y & kSlotIndexMask;
        const unsigned ms = __match_any_sync(0xffffffffu, have ? ss_ : 0xffffffffu);
        if (have && lane == __ffs(ms) - 1) atomicAdd(&hist[ss_], __popc(ms));
        const unsigned md = __match_any_sync(0xffffffffu, have ? ds_ : 0xffffffffu);
        if (have && lane == __ffs(md) - 1) atomicAdd(&hist[n_slots + ds_], __popc(md));
    };
    if (fhave) {
        uint64_t size;
        uint32_t ds, ss;
        if (resolve(flo, fhi, cache, a.slots, n_slots, ds, ss, dst, src, size) == 0 && size <= kSmallMax) sz32 = (unsigned)size;
    }
    if (lazy) count_ticket(fhave, flo);
    unsigned long long sync = 0;
    if (a.skip_barrier) {
        // host-validated table without large descriptors: nothing to agree on, nothing to wait for
        if (tid == 0) sh_first1 = static_end + base1;
        __syncthreads();
    } else {
        // only CTAs that validated a tile have anything to say: the others wait for the verdict
        // without arriving (a 256-descriptor batch is a barrier of one arrival, not 296)
        const unsigned arrivals = min((unsigned)gridDim.x, (n + kThreads - 1) / kThreads);
        const int cta_bad = __syncthreads_or(bad_seen);
        const int cta_chunks = __syncthreads_or(wrote_chunks);
        if (tid == 0 && blockIdx.x < arrivals) {
            const unsigned long long vote = sh_small[1] != 0 && sh_small[0] <= (unsigned long long)(kTeamMax / 16) * sh_small[1];
            const unsigned long long word = 1ull | ((unsigned long long)(cta_bad != 0) << kSyncBadShift) | (vote << kSyncVoteShift);
            // the arrival releases what the other CTAs will read after the barrier: this CTA's chunk-queue
            // items.  A CTA that wrote none has nothing to release (its verdict and vote travel in the word
            // itself), and a relaxed add spares it the fence of a release
            if (cta_chunks) atom_add_release_u64(&ctl->sync, word);
            else asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(&ctl->sync), "l"(word) : "memory");
        }
        // While the barrier fills, the sources of the first descriptors this warp will copy start
        // moving into L2, one 128-byte line per lane: the DRAM would otherwise idle until the
        // barrier is through, and reading a source range that passed its own checks has no
        // effect if the batch is rejected.  Issued AFTER the arrival: a release waits for the
        // prefetches in flight before it.
        unsigned pm = __ballot_sync(0xffffffffu, sz32 != 0 && (unsigned)lane < kPrefetchDescs);
        while (pm) {
            const int l = __ffs(pm) - 1;
            pm &= pm - 1;
            const uint64_t s0 = __shfl_sync(0xffffffffu, src, l), s1 = s0 + __shfl_sync(0xffffffffu, sz32, l);
            for (uint64_t line = (s0 & ~127ull) + 128ull * lane; line < s1; line += 128ull * 32) prefetch_l2_line(line);
        }
        if (tid == 0) {
            unsigned long long v;
            while (((v = ld_acquire(&ctl->sync)) & kSyncFieldMask) < arrivals) {}
            sh_sync = v;
            sh_first1 = static_end + base1;
        }
        __syncthreads();
        sync = sh_sync;
    }
    // the CTA's histogram into the cumulative counters: one atomic per touched slot
    auto flush_hist = [&]() {
        for (uint32_t s = tid; s < 2 * n_slots; s += kThreads) {
            const unsigned v = hist[s];
            if (!v) continue;
            const uint32_t row = s < n_slots ? s : s - n_slots;
            atomicAdd(s < n_slots ? &a.cnt[row].sent : &a.cnt[row].recv, (unsigned long long)v);
            // a message on a global slot also counts at the slot's owner (published by the last CTA)
            if (a.any_global && (slot_row(cache, a.slots, n_slots, row).meta & kRowGlobal))
                atomicAdd(s < n_slots ? &a.gdelta[row].sent : &a.gdelta[row].recv, (unsigned long long)v);
        }
    };
    const bool ok = ((sync >> kSyncBadShift) & kSyncFieldMask) == 0;
    if (blockIdx.x == 0 && tid == 0) ctl->t_mid = globaltimer();

    if (ok) {
        // ============================================================ counters (a6)
        if (use_hist) {
            if (!lazy) flush_hist();
        } else {
            // slot table too large for the shared-memory histogram: count straight into the
            // cumulative counters, now that the batch is known to be valid
            for (uint64_t tile = (uint64_t)blockIdx.x * kThreads; tile < a.n; tile += (uint64_t)gridDim.x * kThreads) {
                const uint64_t i = tile + tid;
                uint32_t ss = 0xffffffffu, ds = 0xffffffffu;
                if (i < a.n) {
                    const uint4 lo = __ldg(reinterpret_cast<const uint4 *>(a.descs + i));
                    ds = lo.x & kSlotIndexMask;
                    ss = lo.y & kSlotIndexMask;
                }
                const unsigned ms = __match_any_sync(0xffffffffu, ss);
                if (i < a.n && lane == __ffs(ms) - 1) {
                    atomicAdd(&a.cnt[ss].sent, (unsigned long long)__popc(ms));
                    if (a.any_global && (slot_row(cache, a.slots, n_slots, ss).meta & kRowGlobal))
                        atomicAdd(&a.gdelta[ss].sent, (unsigned long long)__popc(ms));
                }
                const unsigned md = __match_any_sync(0xffffffffu, ds);
                if (i < a.n && lane == __ffs(md) - 1) {
                    atomicAdd(&a.cnt[ds].recv, (unsigned long long)__popc(md));
                    if (a.any_global && (slot_row(cache, a.slots, n_slots, ds).meta & kRowGlobal))
                        atomicAdd(&a.gdelta[ds].recv, (unsigned long long)__popc(md));
                }
            }
        }

        // ============================================================ phase B1 (a5): CTA per chunk
        // Dynamic tickets, one atomic per CTA per chunk.  Thread 0 runs two rounds ahead: while
        // chunk i is copied, the queue item of chunk i+1 is on its way from L2 and the atomic of
        // chunk i+2 is in flight, so neither latency sits between two chunks (a 32 KiB chunk is
        // about 3 us of copying; the item fetch alone was 0.7 us of it).
        const unsigned n_chunk = (unsigned)(sync >> kSyncChunkShift);
        if (n_chunk) {
            unsigned t1 = 0;          // thread 0: ticket of the next round
            if (tid == 0) {
                const unsigned t0 = atomicAdd(&ctl->ticket, 1u);
                t1 = atomicAdd(&ctl->ticket, 1u);
                sh_ticket[0] = t0;
                if (t0 < n_chunk) sh_item[0] = load_item(a.chunk_q + t0);
            }
            __syncthreads();
            int par = 0;
            while (true) {
                const unsigned t = sh_ticket[par];
                if (t >= n_chunk) break;
                const WorkItem w = sh_item[par];
                unsigned t2 = 0;
                WorkItem nw_item;
                nw_item.src = nw_item.dst = nw_item.size = nw_item.pad = 0;
                if (tid == 0) {
                    t2 = atomicAdd(&ctl->ticket, 1u);
                    if (t1 < n_chunk) nw_item = load_item(a.chunk_q + t1);
                }
                unsigned char *d = reinterpret_cast<unsigned char *>(w.dst);
                const unsigned char *s = reinterpret_cast<const unsigned char *>(w.src);
                if (((w.src | w.dst | w.size) & 15) == 0 && w.size >= a.tma_min) {
                    if (lane == 0) tma_copy_pieces(tma, d, s, w.size, warp, kWarps);
                    __syncwarp();
                } else {
                    copy_span<kUnroll, kLdDefault, uint32_t, kUnrollShifted>(d, s, (uint32_t)w.size, tid, kThreads);
                }
                if (tid == 0) {
                    sh_ticket[par ^ 1] = t1;
                    sh_item[par ^ 1] = nw_item;
                    t1 = t2;
                }
                __syncthreads();
                par ^= 1;
            }
        }

        // ============================================================ phase B2 (a4): warp per small descriptor
        // Small descriptors are read from the table in place.  Each warp takes tickets of
        // `cnt` consecutive descriptors (one per lane) by guided self-scheduling: a ticket is
        // 1/(gss x warps) of what is left, at most 32 and at least 1, so the last tickets are
        // single descriptors.  (Handing the last descriptors out in quarters to shorten the
        // tail measured 3-10 us SLOWER on config 2: a ticket costs an atomic and a descriptor
        // fetch, about 2 us of latency, and three of them in flight per warp do not cover a
        // 1 KiB copy.)  Three tickets are in flight per warp: k is
        // being copied, the descriptors of k+1 are being loaded, the atomic of k+2 is on its
        // way, so neither latency is exposed between two copies.
        first1 = sh_first1 + warp * cnt1;
        // Team-sized descriptors (the CTAs' votes, or the host's own count) are latency-bound, not
        // bandwidth-bound: equal counts are balanced enough, and 2368 warps drawing tickets from
        // one cursor would serialise on it (measured: 5-10 us per batch of 65,536).  They are
        // handed out statically: after its first ticket warp g owns the g-th share of the rest.
        const unsigned voters = min((unsigned)gridDim.x, (n + kThreads - 1) / kThreads);
        const bool static_mode = a.hand_out == kHandOutVote ? 2 * (unsigned)((sync >> kSyncVoteShift) & kSyncFieldMask) >= voters
                                                            : a.hand_out == kHandOutStatic;
        unsigned cur = 0, my_hi = 0;
        if (static_mode) {
            const unsigned rest = n - min(n, static_end), share = (rest + nw - 1) / nw;
            cur = min(n, static_end + (blockIdx.x * kWarps + warp) * share);
            my_hi = min(n, cur + share);
            cnt1 = min(32u, my_hi - cur);
            first1 = cnt1 ? cur : n;
            cur += cnt1;
        }
        uint4 nlo = make_uint4(0, 0, 0, 0), nhi = nlo;
        bool nhave = (unsigned)lane < cnt1 && first1 + lane < n;
        if (nhave) load_desc_raw(a.descs + first1 + lane, nlo, nhi);
        while (first0 < n) {
            unsigned first2 = 0, cnt2 = 0;
            if (static_mode) {
                cnt2 = min(32u, my_hi - cur);
                first2 = cnt2 ? cur : n;
                cur += cnt2;
            } else if (lane == 0) {
                cnt2 = ticket_size(n, first1 + cnt1);
                first2 = static_end + atomicAdd(&ctl->next_desc, cnt2);
            }
            // descriptors of at most kTeamMax bytes: 32 / kTeam of them at a time, each by a team of
            // kTeam lanes, so that their load latencies overlap instead of adding up (config 4:
            // 28 descriptors of 132 B per warp, one after the other, were 1.2 us each)
            const bool tiny = sz32 != 0 && sz32 <= kTeamMax;
            const unsigned tm = __ballot_sync(0xffffffffu, tiny);
            if (tm) {
                if (tiny) sh_rank[warp][__popc(tm & ((1u << lane) - 1u))] = (unsigned char)lane;
                __syncwarp();
                const unsigned cnt = __popc(tm), team = lane / kTeam;
                for (unsigned r0 = 0; r0 < cnt; r0 += 32 / kTeam) {
                    const unsigned r = r0 + team;
                    const int l = r < cnt ? sh_rank[warp][r] : 0;
                    const uint64_t s0 = __shfl_sync(0xffffffffu, src, l);
                    const uint64_t d0 = __shfl_sync(0xffffffffu, dst, l);
                    const unsigned z = __shfl_sync(0xffffffffu, sz32, l);
                    copy_team<kTeam, kTeamVecs>(reinterpret_cast<unsigned char *>(d0), reinterpret_cast<const unsigned char *>(s0),
                                     r < cnt ? z : 0u, lane % kTeam);
                }
                __syncwarp();
            }
            unsigned m = __ballot_sync(0xffffffffu, sz32 > kTeamMax);
            while (m) {
                const int l = __ffs(m) - 1;
                m &= m - 1;
                const uint64_t s0 = __shfl_sync(0xffffffffu, src, l);
                const uint64_t d0 = __shfl_sync(0xffffffffu, dst, l);
                const unsigned z = __shfl_sync(0xffffffffu, sz32, l);
                unsigned char *d = reinterpret_cast<unsigned char *>(d0);
                const unsigned char *s = reinterpret_cast<const unsigned char *>(s0);
                // 16 B vector loads and stores for every alignment; for spans this short the bulk
                // path measured slower and erratic (one driver lane per warp, S5)
                copy_span<kUnroll, kLdDefault, uint32_t, kUnrollShifted>(d, s, z, lane, 32);
            }
            // rotate: k+1 becomes current (its descriptors have landed), k+2 starts loading
            sz32 = nhave ? resolve_small(nlo, nhi, cache, a.slots, n_slots, dst, src) : 0u;
            if (lazy) count_ticket(nhave, nlo);
            first0 = first1;
            first1 = __shfl_sync(0xffffffffu, first2, 0);
            cnt1 = __shfl_sync(0xffffffffu, cnt2, 0);
            nhave = (unsigned)lane < cnt1 && first1 + lane < n;
            if (nhave) load_desc_raw(a.descs + first1 + lane, nlo, nhi);
        }
        if (lane == 0) tma_drain(tma);
    }

    // ================================================================ finish (feeds a7)
    __syncthreads();
    if (lazy) {   // every warp has counted the tickets it copied
        flush_hist();
        __syncthreads();
    }
    if (tid == 0) {
        sh_flag = atom_inc_acq_rel_u32(&ctl->done) == gridDim.x - 1;
        if (sh_flag) sh_seq = __ldcg(&ctl->seq) + 1;   // batches of a context run one after the other: one writer
    }
    __syncthreads();
    if (!sh_flag) return;
    const unsigned long long seq = sh_seq;
    const uint32_t flag = rec_flag(seq);
    unsigned long long *rec = a.rec_ring[(seq - 1) % kRecRing].w;
    // last CTA: every CTA's copies and counter updates are complete and visible on the device
    // (release increments above, acquired by this CTA's thread 0 and handed on by the barrier).
    // Global Memory Slots: what this batch moved from / into a global slot is complete, so it now counts
    // at the slot's owner -- data first (system scope: the owner may be another GPU), then the owner's
    // counters, which is what lets the owner's fence wait for "the expected number of incoming and
    // outgoing data transfers" without a message from this instance.
    if (a.any_global) {
        for (uint32_t s = tid; s < n_slots; s += kThreads) {
            const uint64_t g = __ldcg(a.gptr + s);
            if (!g) continue;
            const unsigned long long sv = __ldcg(&a.gdelta[s].sent), rv = __ldcg(&a.gdelta[s].recv);
            if (!(sv | rv)) continue;
            __threadfence_system();
            SlotCnt *owner = reinterpret_cast<SlotCnt *>(g);
            if (sv) atomicAdd_system(&owner->sent, sv);
            if (rv) atomicAdd_system(&owner->recv, rv);
            a.gdelta[s].sent = 0;
            a.gdelta[s].recv = 0;
        }
    }
    // Publish the cumulative counters and the completion record as flagged 8-byte words.
    for (uint32_t s = tid; s < a.n_push; s += kThreads) {
        const unsigned long long sv = __ldcg(&a.cnt[s].sent), rv = __ldcg(&a.cnt[s].recv);
        unsigned long long *w = a.push + (size_t)s * kPushWordsPerSlot;
        put_word(w + 0, (uint32_t)sv, flag);
        put_word(w + 1, (uint32_t)(sv >> 32), flag);
        put_word(w + 2, (uint32_t)rv, flag);
        put_word(w + 3, (uint32_t)(rv >> 32), flag);
    }
    if (tid == 0) {
        const unsigned long long bad = __ldcg(&ctl->bad_inv), t0 = __ldcg(&ctl->t_start), t1 = __ldcg(&ctl->t_mid),
                                 t2 = globaltimer();
        put_word(rec + kRwBadLo, (uint32_t)bad, flag);
        put_word(rec + kRwBadHi, (uint32_t)(bad >> 32), flag);
        put_word(rec + kRwNChunk, (uint32_t)(sync >> kSyncChunkShift), flag);
        put_word(rec + kRwTStartLo, (uint32_t)t0, flag);
        put_word(rec + kRwTStartHi, (uint32_t)(t0 >> 32), flag);
        put_word(rec + kRwTMidLo, (uint32_t)t1, flag);
        put_word(rec + kRwTMidHi, (uint32_t)(t1 >> 32), flag);
        put_word(rec + kRwTEndLo, (uint32_t)t2, flag);
        put_word(rec + kRwTEndHi, (uint32_t)(t2 >> 32), flag);
        // self-clean: the next batch on the stream finds an all-zero control block
        ctl->seq = seq;
        ctl->bad_inv = 0;
        ctl->sync = 0;
        ctl->ticket = 0;
        ctl->next_desc = 0;
        ctl->done = 0;
    }
}

static int ensure_queues(hicr_ctx *ctx, uint64_t n)
{
    // (while a chain is being recorded nothing may synchronise the stream: hicr_graph_begin sized the queue)
    // With pairwise-disjoint destinations (the epoch precondition) a batch expands into
    // at most 2 n + registered_bytes / kChunkBytes chunks (a first and a last partial one
    // per descriptor).
    const uint64_t need = 2 * n + ctx->registered_bytes / kChunkBytes + 64;
    if (need > ctx->chunk_cap) {
        if (need > kMaxChunks || ctx->capturing) return HICR_ERR_NO_CAPACITY;
        uint64_t cap = std::min(std::max(need, ctx->chunk_cap * 2), kMaxChunks);
        HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (ctx->d_chunk) HICR_CUDA(ctx, cudaFree(ctx->d_chunk));
        ctx->d_chunk = nullptr;
        ctx->chunk_cap = 0;
        HICR_CUDA(ctx, cudaMalloc(&ctx->d_chunk, cap * sizeof(WorkItem)));
        ctx->chunk_cap = cap;
        ctx->queue_version++;   // recorded chains name the old queue: hicr_graph_launch refuses them
    }
    return HICR_OK;
}

static int get_stage(hicr_ctx *ctx, size_t bytes, StageBlock *out)
{
    for (size_t k = 0; k < ctx->free_stage.size(); k++) {
        if (ctx->free_stage[k].bytes >= bytes) {
            *out = ctx->free_stage[k];
            ctx->free_stage.erase(ctx->free_stage.begin() + k);
            return HICR_OK;
        }
    }
    StageBlock b;
    b.bytes = std::max<size_t>(bytes, 1 << 20);
    HICR_CUDA(ctx, cudaHostAlloc(&b.host, b.bytes, cudaHostAllocMapped | cudaHostAllocPortable));
    cudaError_t e = cudaMalloc(&b.dev, b.bytes);
    if (e != cudaSuccess) {
        cudaFreeHost(b.host);
        return cuda_fail(ctx, e, "cudaMalloc(stage)");
    }
    *out = b;
    return HICR_OK;
}

size_t engine_smem_bytes(uint32_t n_slots)
{
    return kSmemStages + kSmemCache + (n_slots <= kSmemSlotHist ? 2 * (size_t)n_slots * sizeof(unsigned) : 0);
}

// Co-resident CTAs of the engine kernel (what a cooperative launch may use).
int engine_setup(hicr_ctx *ctx)
{
    int per_sm = 0;
    HICR_CUDA(ctx, cudaFuncSetAttribute(engine_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)engine_smem_bytes(kSmemSlotHist)));
    HICR_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, engine_kernel, kThreads,
                                                                 engine_smem_bytes(kSmemSlotHist)));
    if (per_sm < 1) return HICR_ERR_NO_CAPACITY;
    per_sm = std::min(per_sm, kCtasPerSm);
    // HICR_TMA_MIN: smallest 16 B-aligned chunk that takes the bulk-copy path (0xffffffff = never).
    // The one tuning knob left; tests run the large-descriptor cases with the path forced on and off.
    const char *e = getenv("HICR_TMA_MIN");
    if (e && *e) ctx->tma_min = (uint32_t)strtoul(e, nullptr, 0);
    if (ctx->tma_min < 16) ctx->tma_min = 16;
    ctx->engine_grid = (int)std::min<unsigned>(ctx->num_sms * per_sm, kMaxGrid);
    return HICR_OK;
}

// ---- launching the engine kernel.  A one-node CUDA graph that is already instantiated starts
// about 3 us sooner than the same cooperative launch through cudaLaunchCooperativeKernel (config 2:
// 97.7 against 100.4-101.2 us per step; the front end replays a command buffer it has seen), so the
// context keeps a few instantiated one-kernel graphs, looks the launch up by its arguments, and
// rewrites the node's parameters of the least recently used one when none matches.  Nothing about
// the batch is cached: every launch runs validation, binning, copies and counters.
constexpr int kLaunchSlots = 8;
struct LaunchSlot {
    NodeLauncher node;
    EngineArgs args;
    unsigned grid = 0;
    size_t smem = 0;
    uint64_t used = 0;
};
struct LaunchCache {
    LaunchSlot slot[kLaunchSlots];
    uint64_t clock = 0;
    bool broken = false;   // the graph path was refused once: stream launches from then on
};

void launch_cache_free(hicr_ctx *ctx)
{
    LaunchCache *c = static_cast<LaunchCache *>(ctx->launch_cache);
    if (!c) return;
    for (auto &s : c->slot) node_free(s.node);
    delete c;
    ctx->launch_cache = nullptr;
}

static cudaError_t launch_engine(hicr_ctx *ctx, EngineArgs &a, unsigned grid, size_t smem)
{
    void *args[] = {&a};
    if (!ctx->launch_cache) {
        // all slots are instantiated now (about 50 us each, once per context), so that a launch that
        // matches none of them later costs a parameter rewrite, not an instantiation
        LaunchCache *fresh = new LaunchCache();
        for (auto &s : fresh->slot)
            if (!fresh->broken && node_prepare(s.node, (const void *)engine_kernel, dim3(grid), dim3(kThreads), smem, args, true, false) !=
                                      cudaSuccess)
                fresh->broken = true;
        ctx->launch_cache = fresh;
    }
    LaunchCache *c = static_cast<LaunchCache *>(ctx->launch_cache);
    if (!c->broken) {
        LaunchSlot *hit = nullptr, *lru = &c->slot[0];
        for (auto &s : c->slot) {
            if (s.node.exec && s.grid == grid && s.smem == smem && memcmp(&s.args, &a, sizeof(EngineArgs)) == 0) hit = &s;
            if (s.used < lru->used) lru = &s;
        }
        LaunchSlot *use = hit ? hit : lru;
        cudaError_t e = node_launch(use->node, (const void *)engine_kernel, dim3(grid), dim3(kThreads), smem, args, true, !hit,
                                    ctx->stream);
        if (e == cudaSuccess) {
            memcpy(&use->args, &a, sizeof(EngineArgs));
            use->grid = grid;
            use->smem = smem;
            use->used = ++c->clock;
            return e;
        }
        c->broken = true;
    }
    return cudaLaunchCooperativeKernel((const void *)engine_kernel, dim3(grid), dim3(kThreads), args, smem, ctx->stream);
}

}  // namespace hicr

using namespace hicr;

extern "C" int hicr_memcpy_batch(hicr_ctx_t *ctx, const hicr_desc_t *descs, uint64_t n, int descs_on_device,
                                 uint64_t *first_bad)
{
    if (!ctx || (!descs && n)) return HICR_ERR_INVALID_ARG;
    if (n == 0) return HICR_OK;
    if (n >= (1ull << 31)) return HICR_ERR_NO_CAPACITY;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));

    if (ctx->capturing) {
        // recorded, not executed: only what the replay can do again -- a device-resident table
        if (!descs_on_device) return HICR_ERR_INVALID_ARG;
        if (ctx->captured_batches == kRecRing) return HICR_ERR_NO_CAPACITY;
    }
    // before anything of this batch is staged: an epoch that has used up its completion records
    // drains them (and recycles the staging blocks of the batches that are then complete)
    if (!ctx->capturing && ctx->batches_in_epoch == kRecRing) {
        int rc = drain_epoch(ctx, false);
        if (rc != HICR_OK) return rc;
    }
    int rc = ensure_queues(ctx, n);
    if (rc != HICR_OK) return rc;

    uint64_t units = ~0ull;   // work tickets of the copy phase, when the host knows them
    const hicr_desc_t *d_descs = descs;
    bool skip_barrier = false;
    uint32_t hand_out = kHandOutVote;
    if (!descs_on_device) {
        // (a2) host-resident table: validated on the host (hicr_stage.cu), all-or-nothing, lowest
        // bad index.  One pass checks a descriptor and copies it into pinned staging, on a few
        // host threads; finished prefixes travel to the device while the rest is being checked.
        // A bad descriptor leaves earlier pieces in the staging block, which nothing reads: no
        // kernel is launched.
        StageBlock b;
        rc = get_stage(ctx, n * sizeof(hicr_desc_t), &b);
        if (rc != HICR_OK) return rc;
        uint64_t ns = 0, nc = 0, small_bytes = 0;
        int bad_status = HICR_OK;
        rc = stage_table(ctx, descs, n, b, first_bad, &bad_status, &nc, &ns, &small_bytes);
        if (rc == HICR_OK && bad_status != HICR_OK) rc = bad_status;
        if (rc != HICR_OK) {
            // earlier pieces of the table may be on their way to b.dev: the block is reusable once they
            // have landed (the error path is not a hot one)
            (void)cudaStreamSynchronize(ctx->stream);
            ctx->free_stage.push_back(b);
            return rc;
        }
        units = nc + (ns + kWarps - 1) / kWarps;
        ctx->used_stage.push_back(b);
        // pinned staging is device-accessible under unified addressing: short tables stay there
        d_descs = static_cast<const hicr_desc_t *>(table_read_in_place(descs, n) ? b.host : b.dev);
        // checked against the host mirror of the slot table, which the device copy follows in
        // stream order: with no chunk queue to wait for either, the kernel needs no barrier
        skip_barrier = nc == 0;
        hand_out = ns && small_bytes <= kTeamMax * ns ? kHandOutStatic : kHandOutDynamic;
    }

    EngineArgs a;
    memset(&a, 0, sizeof(a));   // (padding included: launches are looked up by these bytes)
    a.descs = d_descs;
    a.n = n;
    a.slots = ctx->d_slots;
    a.n_slots = (uint32_t)ctx->rows.size();
    a.tma_min = ctx->tma_min;
    a.ctl = ctx->d_ctl;
    a.chunk_q = ctx->d_chunk;
    a.chunk_cap = ctx->chunk_cap;
    a.cnt = ctx->d_cnt;
    a.rec_ring = ctx->d_rec;
    a.push = ctx->d_rec[kRecRing].w;
    a.n_push = std::min<uint32_t>(a.n_slots, kPushSlots);
    a.skip_barrier = skip_barrier ? 1u : 0u;
    a.hand_out = hand_out;
    a.gptr = ctx->d_gptr;
    a.gdelta = ctx->d_gdelta;
    a.any_global = ctx->n_global ? 1u : 0u;

    // grid: every co-resident CTA unless the host knows the batch is smaller than that
    uint64_t want = std::max<uint64_t>((n + kThreads - 1) / kThreads, units == ~0ull ? (uint64_t)ctx->engine_grid : units);
    const unsigned grid = (unsigned)std::max<uint64_t>(1, std::min<uint64_t>(want, (uint64_t)ctx->engine_grid));
    void *args[] = {&a};
    if (ctx->capturing) {
        HICR_CUDA(ctx, cudaLaunchCooperativeKernel((const void *)engine_kernel, dim3(grid), dim3(kThreads), args,
                                                   engine_smem_bytes(a.n_slots), ctx->stream));
        ctx->captured_batches++;
        return HICR_OK;   // the context's books are kept by hicr_graph_launch
    }
    if (ctx->profiling) HICR_CUDA(ctx, cudaEventRecord(ctx->ev[0], ctx->stream));
    HICR_CUDA(ctx, launch_engine(ctx, a, grid, engine_smem_bytes(a.n_slots)));
    ctx->launches++;
    if (ctx->profiling) {
        HICR_CUDA(ctx, cudaEventRecord(ctx->ev[1], ctx->stream));
        ctx->ev_valid = true;
    }
    ctx->batch_seq++;
    ctx->batches_in_epoch++;
    ctx->epoch_open = true;
    ctx->last_n_push = a.n_push;
    ctx->push_stale = false;
    return HICR_OK;
}

// ---------------------------------------------------------------- replayable chains (hicr_graph_*)
struct hicr_graph {
    hicr_ctx *ctx = nullptr;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    uint32_t n_batches = 0, n_push = 0;
    uint64_t table_version = 0, queue_version = 0;
};

extern "C" int hicr_graph_begin(hicr_ctx_t *ctx, uint64_t max_descs_per_batch)
{
    if (!ctx || max_descs_per_batch >= (1ull << 31)) return HICR_ERR_INVALID_ARG;
    if (ctx->capturing) return HICR_ERR_BUSY;
    if (!ctx->stream) return HICR_ERR_INVALID_ARG;   // the legacy default stream cannot be captured
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    int rc = ensure_queues(ctx, max_descs_per_batch);
    if (rc != HICR_OK) return rc;
    HICR_CUDA(ctx, cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeRelaxed));
    ctx->capturing = true;
    ctx->captured_batches = 0;
    return HICR_OK;
}

extern "C" int hicr_graph_end(hicr_ctx_t *ctx, hicr_graph_t **out)
{
    if (!ctx || !out) return HICR_ERR_INVALID_ARG;
    *out = nullptr;
    if (!ctx->capturing) return HICR_ERR_INVALID_ARG;
    ctx->capturing = false;
    hicr_graph *g = new hicr_graph();
    g->ctx = ctx;
    g->n_batches = ctx->captured_batches;
    g->n_push = std::min<uint32_t>((uint32_t)ctx->rows.size(), kPushSlots);
    g->table_version = ctx->table_version;
    g->queue_version = ctx->queue_version;
    cudaError_t e = cudaStreamEndCapture(ctx->stream, &g->graph);
    if (e == cudaSuccess && g->graph) e = cudaGraphInstantiate(&g->exec, g->graph, 0);
    if (e != cudaSuccess || !g->graph) {
        if (g->graph) cudaGraphDestroy(g->graph);
        delete g;
        return cuda_fail(ctx, e == cudaSuccess ? cudaErrorUnknown : e, "hicr_graph_end");
    }
    *out = g;
    return HICR_OK;
}

extern "C" int hicr_graph_launch(hicr_graph_t *g)
{
    if (!g) return HICR_ERR_INVALID_ARG;
    hicr_ctx *ctx = g->ctx;
    if (ctx->capturing) return HICR_ERR_BUSY;
    if (g->table_version != ctx->table_version) return HICR_ERR_INVALID_ARG;   // the recorded launches name another slot table
    if (g->queue_version != ctx->queue_version) return HICR_ERR_INVALID_ARG;   // ... or a chunk queue that has been freed since
    if (g->n_batches == 0) return HICR_OK;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    if (ctx->batches_in_epoch + g->n_batches > (uint32_t)kRecRing) {
        int rc = drain_epoch(ctx, false);
        if (rc != HICR_OK) return rc;
    }
    HICR_CUDA(ctx, cudaGraphLaunch(g->exec, ctx->stream));
    ctx->launches += g->n_batches;
    ctx->batch_seq += g->n_batches;
    ctx->batches_in_epoch += g->n_batches;
    ctx->epoch_open = true;
    ctx->last_n_push = g->n_push;
    ctx->push_stale = false;
    return HICR_OK;
}

extern "C" int hicr_graph_destroy(hicr_graph_t *g)
{
    if (!g) return HICR_ERR_INVALID_ARG;
    (void)cudaStreamSynchronize(g->ctx->stream);
    if (g->exec) cudaGraphExecDestroy(g->exec);
    if (g->graph) cudaGraphDestroy(g->graph);
    (void)cudaGetLastError();
    delete g;
    return HICR_OK;
}
