// hicr_internal.cuh -- shared declarations of the sm_100a copy engine (not installed).
//
// Layout of the device-side state, the work-item formats produced by the binning
// kernel, and the one copy routine (copy_span) every data-moving kernel uses.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>
#include <vector>

#include "../../include/hicr.h"

namespace hicr {

// ---------------------------------------------------------------- tunables / classes
// 0 < size <= kSmallMax : copied in place from the descriptor table, warp per descriptor (a4)
// size >  kSmallMax     : split at kChunkBytes-aligned destination addresses, CTA-per-chunk queue (a5)
constexpr uint64_t kSmallMax = 8192;
constexpr uint64_t kChunkBytes = 131072;   // 128 KiB.  Config 3a: 32 KiB chunks 5765 GB/s, 64 KiB 5990, 128 KiB 6118 (fewer CTA barriers and tickets per byte)
constexpr int kThreads = 256;              // 8 warps per CTA of the engine kernel
constexpr int kWarps = kThreads / 32;
constexpr int kCtasPerSm = 2;              // persistent grid = SMs x kCtasPerSm; 16 warps x 4 x 16 B x 32 lanes = 32 KiB of
                                           // loads in flight per SM is where a 4 KiB page copy peaks on B200 (S5)
constexpr int kUnroll = 4;                 // 16-byte vectors in flight per lane (aligned source)
constexpr int kUnrollShifted = 8;          // the same for byte-shifted sources
constexpr uint32_t kSmemSlotHist = 1024;   // per-CTA shared-memory counter histogram up to this many slots
constexpr uint32_t kSlotCache = 256;       // slot-table rows cached in shared memory (larger tables are read from L2)
constexpr uint32_t kTmaPiece = 4096;       // bytes per bulk copy
constexpr int kTmaStages = 2;              // shared-memory stages per warp: load of piece k overlaps the store of piece k-1
constexpr uint32_t kTmaMinDefault = 1024;  // aligned spans of at least this many bytes take the TMA bulk path
constexpr int kRecRing = 64;               // host completion records (= batches per epoch before an internal drain)
constexpr uint32_t kPushSlots = 256;       // counters of the first kPushSlots slots are pushed into the record area
constexpr int kTeam = 4;                   // lanes per team
constexpr int kTeamVecs = 4;               // 16 B vectors per lane of a team
constexpr unsigned kTeamMax = 16 * kTeam * kTeamVecs;   // descriptors up to this size (256 B) are copied by teams, 32 / kTeam at a time
constexpr uint64_t kZeroCopyDescs = 1024;   // host tables up to this many descriptors are read by the kernel straight from
                                            // pinned staging (32 KiB over PCIe costs less than enqueueing a copy: ~1.5 vs ~5 us)
constexpr unsigned kMaxGroup = 32;         // units per warp ticket, at most (one per lane)
constexpr unsigned kGss = 3;               // guided self-scheduling: a warp ticket is 1 / (kGss x warps) of what is left
constexpr unsigned kPrefetchDescs = 2;     // descriptors per warp whose source goes to L2 while the grid barrier fills
constexpr int kStageThreadsMax = 8;        // host threads that check and stage a host-resident table (caller included):
                                           // half the cores the process may use, at most this many (4 threads: 92 us for the
                                           // 2 MiB table of config 2, bound by host memory bandwidth)

// error ids packed into Ctl::bad (lower id does not mean higher priority; index decides)
constexpr unsigned kBadInvalidSlot = 1, kBadOutOfBounds = 2, kBadNoCapacity = 3, kBadDirection = 4;

// A slot id is {generation:20 | table index:12}.  Unregistering frees the index; the next
// registration that takes it bumps the generation, so an id kept from before names nothing.
constexpr int kSlotIndexBits = 12;
constexpr uint32_t kSlotIndexMask = (1u << kSlotIndexBits) - 1;
static_assert((1u << kSlotIndexBits) == HICR_MAX_SLOTS, "slot index field covers the table");

// One row of the device slot table: "minimum information required to describe a segment
// of memory (e.g., size, starting address)".
//   meta = {remote:1 | global:1 | generation:18 | size:44}; all ones = not registered.
// global = a Global Memory Slot; remote = its storage belongs to another
// instance (base is then a peer-mapped address).
struct SlotRow {
    uint64_t base;
    uint64_t meta;
};
constexpr int kSizeBits = 44, kGenBits = 18;
constexpr uint64_t kSizeMask = (1ull << kSizeBits) - 1;          // slots of up to 16 TiB - 1
constexpr uint64_t kGenMask = (1ull << kGenBits) - 1;
constexpr uint64_t kRowGlobal = 1ull << 62, kRowRemote = 1ull << 63;
constexpr uint64_t kInvalidMeta = ~0ull;
constexpr uint32_t kMaxGen = (uint32_t)kGenMask - 1;             // an index whose generation reaches this is retired

// Per-slot message counters, cumulative since registration (reading 7).
struct SlotCnt {
    unsigned long long sent, recv;
};

__host__ __device__ inline uint64_t row_size(const SlotRow &r) { return r.meta & kSizeMask; }
__host__ __device__ inline uint32_t row_gen(const SlotRow &r) { return (uint32_t)((r.meta >> kSizeBits) & kGenMask); }
__host__ __device__ inline uint64_t row_meta(uint64_t size, uint32_t gen, uint64_t flags)
{
    return size | ((uint64_t)gen << kSizeBits) | flags;
}

// (a2) THE validator, used by the engine kernel for device-resident tables and by the host
// threads for host-resident ones: one end of a transfer against its slot row.  `in_table` =
// the id's index lies inside the table.  Overflow-safe "off + size <= slot size".
__host__ __device__ inline unsigned check_end(const SlotRow &r, bool in_table, uint32_t id, uint64_t off, uint64_t size)
{
    if (!in_table || r.meta == kInvalidMeta || row_gen(r) != (id >> kSlotIndexBits)) return kBadInvalidSlot;
    const uint64_t sz = row_size(r);
    if (off > sz || size > sz - off) return kBadOutOfBounds;
    return 0;
}
// Whole descriptor: destination before source, then the direction rule -- Local-to-Local,
// Local-to-Global and Global-to-Local are allowed, "Global-to-Global operations are not
// permitted".
__host__ __device__ inline unsigned check_transfer(const SlotRow &dr, bool d_in, uint32_t d_id, uint64_t d_off,
                                                   const SlotRow &sr, bool s_in, uint32_t s_id, uint64_t s_off,
                                                   uint64_t size)
{
    unsigned bad = check_end(dr, d_in, d_id, d_off, size);
    if (bad) return bad;
    bad = check_end(sr, s_in, s_id, s_off, size);
    if (bad) return bad;
    if (dr.meta & sr.meta & kRowGlobal) return kBadDirection;
    return 0;
}

// Item of the chunk queue (32 B so that one lane fetches it with two 16 B loads).
struct __align__(16) WorkItem {
    uint64_t src;
    uint64_t dst;
    uint64_t size;
    uint64_t pad;
};

// Device control block of the engine kernel.  All-zero between batches (but for seq): the last CTA of
// a batch publishes the host record and then clears it, so consecutive batches on the
// stream reuse it without any memset.  Every word that many CTAs hammer with atomics sits
// on its own 128-byte line: 2368 warps taking tickets must not delay the grid barrier or
// the reads that follow it (they did, by up to 3 us, when all of this shared one line).
struct __align__(128) Ctl {
    // line 0: written rarely
    unsigned long long bad_inv;   // atomicMax of ~((index << 4) | error id); 0 = no error
    unsigned long long t_start;   // %globaltimer at kernel start (CTA 0)
    unsigned long long t_mid;     // %globaltimer after the grid barrier (CTA 0)
    unsigned long long seq;       // batches this context has completed; NOT cleared between batches
    unsigned int pad0[24];
    // line 1: the grid barrier between validation/binning and the copies, and everything a
    // CTA must know when it leaves it, in ONE word, so that the poll that sees the last
    // arrival also delivers the verdict (no second L2 round trip after the barrier):
    //   bits  0..11  CTAs arrived              bits 12..23  CTAs that saw an invalid descriptor
    //   bits 24..35  CTAs whose small descriptors are team-sized on average (static hand-out)
    //   bits 36..63  items in the chunk queue
    unsigned long long sync;
    unsigned int pad1[30];
    unsigned int ticket;          // line 2: CTA tickets of the chunk queue
    unsigned int pad2[31];
    unsigned int next_desc;       // line 3: warp tickets, first unit not yet handed out
    unsigned int pad3[31];
    unsigned int done;            // line 4: CTAs that finished the copy phase
    unsigned int pad4[31];
};
constexpr int kSyncBadShift = 12, kSyncVoteShift = 24, kSyncChunkShift = 36;
constexpr unsigned long long kSyncFieldMask = 0xfffull;
constexpr unsigned kMaxGrid = 4095;          // engine grid limit imposed by the 12-bit fields
constexpr uint64_t kMaxChunks = (1ull << 28) - 1;
static_assert(sizeof(Ctl) == 640, "Ctl is five 128-byte lines");

// Completion record of one batch in mapped pinned host memory, written by the last CTA
// and polled by hicr_fence.  Every 8-byte word is {low: 32 bits of payload, high: flag},
// flag = rec_flag(batch sequence number) != 0.  A naturally aligned 8-byte store is
// single-copy atomic, so a word whose flag matches carries its payload: no system-scope
// fence orders the words (each one costs about 1.6 us on the way out, S5.1).
constexpr int kRecWords = 16;
enum RecWord { kRwBadLo = 0, kRwBadHi, kRwNChunk, kRwTStartLo, kRwTStartHi, kRwTMidLo, kRwTMidHi, kRwTEndLo, kRwTEndHi,
               kRwUsed };
struct __align__(128) HostRecord {
    unsigned long long w[kRecWords];
};
static_assert(sizeof(HostRecord) == 128, "HostRecord is 128 bytes");
// pushed counters follow the kRecRing records: 4 words per slot (sent lo, sent hi, recv lo, recv hi)
constexpr int kPushWordsPerSlot = 4;
__host__ __device__ inline uint32_t rec_flag(uint64_t seq) { return (uint32_t)(seq % 0xffffffffull) + 1u; }

// Channel state in device memory; head and tail on separate 128 B lines so the
// producer's and the consumer's polls do not share a line.
struct __align__(128) ChannelState {
    unsigned long long head;     // tokens ever pushed (producer-advanced)
    unsigned long long pad0[15];
    unsigned long long tail;     // tokens ever popped (consumer-advanced)
    unsigned long long pad1[15];
};
static_assert(sizeof(ChannelState) == 256, "ChannelState is two lines");

// One ring of a device-resident pipeline run (hicr_pipe.cu): its counters, the ring slot, and where
// the run's first token comes from and goes to.  count0 = head = tail at entry.
struct PipeRing {
    ChannelState *st;
    unsigned char *ring;
    const unsigned char *src;
    unsigned char *dst;
    unsigned long long count0;
    uint32_t id_ring, id_src, id_dst, pad;   // table indices, for the message counters
};

// Result of one host-call push/pop, written by the kernel into mapped pinned memory.
struct CallResult {
    unsigned long long k, head, tail;
    long long status;
    unsigned long long seq;   // (unused by the kernels; the host keeps the call's sequence number here)
    unsigned long long w[8];  // host-call path: the result as flagged words {flag:32 | payload:32}, polled by the host
};

#ifdef __CUDACC__
// ---------------------------------------------------------------- device helpers
enum LdPolicy { kLdStream = 0, kLdL2 = 1, kLdDefault = 2 };

template <int POL>
__device__ __forceinline__ uint4 ld16(const uint4 *p)
{
    return POL == kLdStream ? __ldcs(p) : POL == kLdL2 ? __ldcg(p) : *p;
}
template <int POL>
__device__ __forceinline__ unsigned char ld1(const unsigned char *p)
{
    return POL == kLdStream ? __ldcs(p) : POL == kLdL2 ? __ldcg(p) : *p;
}
template <int POL>
__device__ __forceinline__ void st16(uint4 *p, uint4 v)
{
    if (POL == kLdStream) __stcs(p, v); else if (POL == kLdL2) __stcg(p, v); else *p = v;
}

// dst vector = 16 bytes starting 4*q + rbits/8 bytes into the 32-byte pair (a, nx); q in 0..3.
__device__ __forceinline__ uint4 shift_combine(const uint4 &a, const uint4 &nx, unsigned q, unsigned rbits)
{
    // five consecutive words starting at word q of {a.x a.y a.z a.w nx.x nx.y nx.z nx.w}
    const bool q1 = q & 1, q2 = q & 2;
    const unsigned e0 = q1 ? a.y : a.x, e1 = q1 ? a.z : a.y, e2 = q1 ? a.w : a.z, e3 = q1 ? nx.x : a.w,
                   e4 = q1 ? nx.y : nx.x, e5 = q1 ? nx.z : nx.y, e6 = q1 ? nx.w : nx.z;
    const unsigned w0 = q2 ? e2 : e0, w1 = q2 ? e3 : e1, w2 = q2 ? e4 : e2, w3 = q2 ? e5 : e3, w4 = q2 ? e6 : e4;
    uint4 o;
    o.x = __funnelshift_r(w0, w1, rbits);
    o.y = __funnelshift_r(w1, w2, rbits);
    o.z = __funnelshift_r(w2, w3, rbits);
    o.w = __funnelshift_r(w3, w4, rbits);
    return o;
}

// Body of a copy whose destination is 16 B-aligned and whose source is `4*q + rbits/8` bytes
// past a 16 B boundary (not both zero).  sA = source rounded down to 16 B.  Each warp
// takes tiles of 32*U consecutive destination vectors; lane l loads aligned source
// vectors l, l+32, ... once, and gets the vector after its own from lane l+1 by shuffle
// (lane 31 from lane 0's next load), so every source byte is requested from L2 once.
template <int U, int POL, typename IDX>
__device__ __forceinline__ void copy_body_shifted(uint4 *__restrict__ d4, const uint4 *__restrict__ sA,
                                                  IDX nvec, unsigned q, unsigned rbits, int lane, int warp,
                                                  int nwarps)
{
    constexpr IDX kTile = 32 * U;
    const IDX nfull = nvec / kTile;
    const int nxt_lane = (lane + 1) & 31;
    for (IDX t = warp; t < nfull; t += nwarps) {
        const IDX base = t * kTile + lane;
        uint4 a[U + 1];
#pragma unroll
        for (int u = 0; u < U; u++) a[u] = ld16<POL>(sA + base + 32 * u);
        a[U] = a[U - 1];
        if (lane == 0) a[U] = ld16<POL>(sA + base + 32 * U);
#pragma unroll
        for (int u = 0; u < U; u++) {
            const uint4 give = lane == 0 ? a[u + 1] : a[u];
            uint4 nx;
            nx.x = __shfl_sync(0xffffffffu, give.x, nxt_lane);
            nx.y = __shfl_sync(0xffffffffu, give.y, nxt_lane);
            nx.z = __shfl_sync(0xffffffffu, give.z, nxt_lane);
            nx.w = __shfl_sync(0xffffffffu, give.w, nxt_lane);
            st16<POL>(d4 + base + 32 * u, shift_combine(a[u], nx, q, rbits));
        }
    }
    const IDX rem0 = nfull * kTile;
    if (rem0 < nvec && warp == (int)(nfull % (IDX)nwarps)) {
        // ragged last tile: vector v is stored if v < nvec; aligned source vector v is
        // loaded if v <= nvec (vector nvec still holds bytes of destination vector nvec-1)
        const IDX base = rem0 + lane;
        uint4 a[U + 1];
#pragma unroll
        for (int u = 0; u < U; u++) {
            a[u] = make_uint4(0, 0, 0, 0);
            if (base + 32 * u <= nvec) a[u] = ld16<POL>(sA + base + 32 * u);
        }
        a[U] = make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int u = 0; u < U; u++) {
            const uint4 give = lane == 0 ? a[u + 1] : a[u];
            uint4 nx;
            nx.x = __shfl_sync(0xffffffffu, give.x, nxt_lane);
            nx.y = __shfl_sync(0xffffffffu, give.y, nxt_lane);
            nx.z = __shfl_sync(0xffffffffu, give.z, nxt_lane);
            nx.w = __shfl_sync(0xffffffffu, give.w, nxt_lane);
            if (base + 32 * u < nvec) st16<POL>(d4 + base + 32 * u, shift_combine(a[u], nx, q, rbits));
        }
    }
}

template <int U, int POL, typename IDX>
__device__ __forceinline__ void copy_body_aligned(uint4 *__restrict__ d4, const uint4 *__restrict__ s4,
                                                  IDX nvec, int lane, int warp, int nwarps)
{
    constexpr IDX kTile = 32 * U;
    const IDX nfull = nvec / kTile;
    for (IDX t = warp; t < nfull; t += nwarps) {
        const IDX base = t * kTile + lane;
        uint4 a[U];
#pragma unroll
        for (int u = 0; u < U; u++) a[u] = ld16<POL>(s4 + base + 32 * u);
#pragma unroll
        for (int u = 0; u < U; u++) st16<POL>(d4 + base + 32 * u, a[u]);
    }
    const IDX rem0 = nfull * kTile;
    if (rem0 < nvec && warp == (int)(nfull % (IDX)nwarps)) {
        const IDX base = rem0 + lane;
        uint4 a[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            a[u] = make_uint4(0, 0, 0, 0);
            if (base + 32 * u < nvec) a[u] = ld16<POL>(s4 + base + 32 * u);
        }
#pragma unroll
        for (int u = 0; u < U; u++)
            if (base + 32 * u < nvec) st16<POL>(d4 + base + 32 * u, a[u]);
    }
}

// dst[i] = src[i], i < n, for any alignment of dst and src.  Called by ALL threads of a
// group of `gsize` threads (a multiple of 32: one warp, or a whole CTA), gtid in
// [0, gsize).  Byte head up to the first 16 B boundary of dst, 16 B vector body with
// aligned stores (aligned or byte-shifted loads), byte tail (a4/a5 of SURVEY.md S8(a)).
// IDX = uint32_t when n < 2^32 is known (fewer registers).  U / US = 16 B vectors in flight per
// lane in the aligned / byte-shifted body.
template <int U, int POL, typename IDX = uint64_t, int US = U>
__device__ __forceinline__ void copy_span(unsigned char *__restrict__ dst, const unsigned char *__restrict__ src,
                                          IDX n, int gtid, int gsize)
{
    const int lane = gtid & 31, warp = gtid >> 5, nwarps = gsize >> 5;
    IDX head = (IDX)((16 - (reinterpret_cast<uintptr_t>(dst) & 15)) & 15);
    if (head > n) head = n;
    if ((IDX)gtid < head) dst[gtid] = ld1<POL>(src + gtid);
    dst += head;
    src += head;
    n -= head;
    const IDX nvec = n >> 4;
    const unsigned tail = (unsigned)(n & 15);
    {
        const unsigned t = (unsigned)(gsize - 1 - gtid);   // the last threads take the tail
        if (t < tail) dst[(size_t)nvec * 16 + t] = ld1<POL>(src + (size_t)nvec * 16 + t);
    }
    if (nvec == 0) return;
    uint4 *d4 = reinterpret_cast<uint4 *>(dst);
    const unsigned s = (unsigned)(reinterpret_cast<uintptr_t>(src) & 15);
    if (s == 0) {
        copy_body_aligned<U, POL, IDX>(d4, reinterpret_cast<const uint4 *>(src), nvec, lane, warp, nwarps);
        return;
    }
    const uint4 *sA = reinterpret_cast<const uint4 *>(src - s);
    copy_body_shifted<US, POL, IDX>(d4, sA, nvec, s >> 2, (s & 3) * 8, lane, warp, nwarps);
}

// dst[i] = src[i], i < n <= 16 * G * V, by a TEAM of G consecutive lanes, tl = lane within the
// team.  The teams of a warp run this together, each on its own short span (n may differ per
// team, 0 included).  Same decomposition as copy_span -- byte head up to the first 16 B
// boundary of dst, aligned 16 B stores with aligned or byte-shifted loads, byte tail -- but
// fully predicated and with EVERY load issued before the first store, so a span costs one
// memory round trip, not one per part.  A shifted destination vector reads the two aligned
// source vectors that hold its bytes (the second is the neighbour lane's first: an L1 hit);
// both contain bytes of the span, so nothing outside the source range's 16 B granules is
// touched.
template <int G, int V>
__device__ __forceinline__ void copy_team(unsigned char *__restrict__ dst, const unsigned char *__restrict__ src,
                                          unsigned n, int tl)
{
    constexpr int HB = (15 + G - 1) / G;   // head / tail bytes per lane, at most
    unsigned head = (16u - (unsigned)(reinterpret_cast<uintptr_t>(dst) & 15)) & 15u;
    if (head > n) head = n;
    const unsigned char *s1 = src + head;
    unsigned char *d1 = dst + head;
    const unsigned n1 = n - head, nvec = n1 >> 4, tail = n1 & 15u;
    const unsigned s = (unsigned)(reinterpret_cast<uintptr_t>(s1) & 15);
    const uint4 *sA = reinterpret_cast<const uint4 *>(s1 - s);
    uint4 *d4 = reinterpret_cast<uint4 *>(d1);
    unsigned char hb[HB], tb[HB];
    uint4 a[V], b[V];
#pragma unroll
    for (int k = 0; k < HB; k++) {
        hb[k] = tb[k] = 0;
        if (tl + G * k < head) hb[k] = src[tl + G * k];
        if (tl + G * k < tail) tb[k] = s1[nvec * 16 + tl + G * k];
    }
#pragma unroll
    for (int k = 0; k < V; k++) {
        a[k] = b[k] = make_uint4(0, 0, 0, 0);
        if (tl + G * k < nvec) {
            a[k] = sA[tl + G * k];
            if (s) b[k] = sA[tl + G * k + 1];
        }
    }
#pragma unroll
    for (int k = 0; k < HB; k++) {
        if (tl + G * k < head) dst[tl + G * k] = hb[k];
        if (tl + G * k < tail) d1[nvec * 16 + tl + G * k] = tb[k];
    }
#pragma unroll
    for (int k = 0; k < V; k++)
        if (tl + G * k < nvec) d4[tl + G * k] = shift_combine(a[k], b[k], s >> 2, (s & 3) * 8);   // s = 0: a[k] itself
}

__device__ __forceinline__ unsigned long long ld_acquire(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
// Release-increment by one thread after a __syncthreads(): the CTA's earlier writes are
// ordered before it (bar.sync + release cumulativity) without the L1 invalidation that
// __threadfence() adds.
__device__ __forceinline__ void red_release_u32(unsigned *p)
{
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(p) : "memory");
}
__device__ __forceinline__ unsigned atom_inc_acq_rel_u32(unsigned *p)
{
    unsigned v;
    asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void atom_add_release_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void st_release(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// ---- 1-D bulk async copies (TMA) through shared memory, completion by mbarrier transaction
// bytes on the way in and by bulk async-groups on the way out.  Addresses and sizes must
// be multiples of 16 bytes.
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    unsigned ok = 0;
    while (!ok) {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
    }
}
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gsrc, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *gdst, const void *smem_src, unsigned bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read_all() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }

// State of one warp's bulk-copy driver (lane 0): a ring of kTmaStages stages of kTmaPiece
// bytes, one mbarrier each.  Piece k is loaded into stage k % kTmaStages while the store
// of piece k-1 is still reading its own stage, so a warp keeps one load and one store in
// flight (measured best at 2 stages x 16 warps per SM for 4 KiB pages, S5).
struct TmaLane {
    unsigned char *stage;   // kTmaStages x kTmaPiece bytes
    uint64_t *bar;          // kTmaStages mbarriers
    unsigned k;             // pieces issued so far
    unsigned char *pend_dst;   // destination of piece k-1, whose store has not been issued yet
    unsigned pend_len;         // 0 = nothing pending
    bool stores;               // any bulk store issued and not yet drained
};

// Driver lane only.  Issue the store of the pending piece (after its load has landed).
__device__ __forceinline__ void tma_store_pending(TmaLane &t)
{
    if (t.pend_len) {
        const unsigned kp = t.k - 1, sp = kp % kTmaStages;
        mbar_wait(t.bar + sp, (kp / kTmaStages) & 1);
        bulk_s2g(t.pend_dst, t.stage + sp * kTmaPiece, t.pend_len);
        bulk_commit();
        t.pend_len = 0;
        t.stores = true;
    }
}

// Driver lane only: one piece of len <= kTmaPiece bytes; dst, src and len multiples of 16.
// Order per piece (the one that measured best, S5): wait for the load of piece
// k-1 and issue its store; wait until at most that one store is still reading shared
// memory (so the stage of piece k-2 is free); issue the load of piece k into it.
__device__ __forceinline__ void tma_piece(TmaLane &t, unsigned char *dst, const unsigned char *src, unsigned len)
{
    const unsigned st = t.k % kTmaStages;
    tma_store_pending(t);
    if (t.stores) bulk_wait_read<kTmaStages - 1>();
    mbar_expect_tx(t.bar + st, len);
    bulk_g2s(t.stage + st * kTmaPiece, src, len, t.bar + st);
    t.pend_dst = dst;
    t.pend_len = len;
    t.k++;
}

// Driver lane only: dst[0, n) = src[0, n) for piece indices first, first + stride, ... of
// kTmaPiece bytes each; dst, src and n are multiples of 16.
__device__ __forceinline__ void tma_copy_pieces(TmaLane &t, unsigned char *dst, const unsigned char *src, uint64_t n,
                                                unsigned first, unsigned stride)
{
    for (uint64_t off = (uint64_t)first * kTmaPiece; off < n; off += (uint64_t)stride * kTmaPiece)
        tma_piece(t, dst + off, src + off, (unsigned)min((uint64_t)kTmaPiece, n - off));
}

// Driver lane only: everything issued so far is written (complete, not only done reading
// shared memory) and ordered before the generic-proxy release that follows.
__device__ __forceinline__ void tma_drain(TmaLane &t)
{
    tma_store_pending(t);
    if (t.stores) {
        bulk_wait_all();
        fence_proxy_async();
        t.stores = false;
    }
}

#endif  // __CUDACC__

// ---------------------------------------------------------------- host-side context
struct StageBlock {
    void *host = nullptr;   // pinned
    void *dev = nullptr;
    size_t bytes = 0;
};

// One instantiated one-kernel CUDA graph: launching it starts the kernel about 3 us sooner than a
// stream launch of the same kernel (measured on config 2 and on the host-call push / pop), and its
// parameters can be rewritten in place (node_launch with update = true).
struct NodeLauncher {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaGraphNode_t node = nullptr;
};
// Launch `func` through the launcher: builds it on first use, rewrites the node's parameters when
// `update`, then cudaGraphLaunch.  A failure to build or update is returned (the caller falls back).
cudaError_t node_prepare(NodeLauncher &l, const void *func, dim3 grid, dim3 block, size_t smem, void **args, bool cooperative,
                         bool update);
cudaError_t node_launch(NodeLauncher &l, const void *func, dim3 grid, dim3 block, size_t smem, void **args, bool cooperative,
                        bool update, cudaStream_t stream);
void node_free(NodeLauncher &l);

class StagePool;
struct GlobalTable;   // hicr_global.cu: the context's Global Memory Slots, by table index and by (tag, key)

}  // namespace hicr

struct hicr_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 0;
    std::string cuda_error;

    // slot table: host mirror + device copy.  rows.size() = high-water mark of indices handed
    // out; a freed index keeps its generation in `gen` and waits in `free_idx` (lowest first).
    std::vector<hicr::SlotRow> rows;         // meta == kInvalidMeta: not registered
    std::vector<uint32_t> gen;               // generation of the current (or last) registration of the index
    std::vector<uint32_t> free_idx;          // freed indices, kept sorted descending (back() = lowest)
    std::vector<hicr::SlotCnt> cnt;          // host mirror of the counters, refreshed at fence / channel calls
    std::vector<uint64_t> born;              // batch_seq when the index was last handed out (older snapshots are not its)
    std::vector<uint32_t> ring_refs;         // live channels using the slot as ring
    hicr::SlotRow *d_slots = nullptr;        // [HICR_MAX_SLOTS]
    hicr::SlotCnt *d_cnt = nullptr;          // [HICR_MAX_SLOTS]
    uint64_t registered_bytes = 0;

    // engine control block (device, self-cleaning) and per-batch completion records
    // (mapped pinned host memory: kRecRing records, then 2 * kPushSlots pushed counters)
    hicr::Ctl *d_ctl = nullptr;
    hicr::HostRecord *h_rec = nullptr;       // host view
    hicr::HostRecord *d_rec = nullptr;       // device alias
    uint64_t batch_seq = 0;                  // sequence number of the last launched batch (1-based)
    uint32_t batches_in_epoch = 0;           // records in use since the last fence (or internal drain)
    uint64_t epoch_batch_base = 0;           // batches drained earlier in this epoch
    bool epoch_open = false;                 // any work enqueued since the last fence
    int epoch_error = HICR_OK;               // first deferred error found so far in this epoch
    uint64_t epoch_error_batch = 0, epoch_error_index = 0;
    int last_error = HICR_OK;                // of the last fence, for hicr_fence_error
    uint64_t last_error_batch = 0, last_error_index = 0;
    uint32_t last_n_push = 0;                // slots whose counters the last launched batch pushes beside its record
    bool push_stale = true;                  // the pushed snapshot of the last batch does not cover everything the mirror
                                             // must show (a channel kernel ran after it, the table changed, ...)

    // chunk queue (large descriptors expanded by the binning phase)
    hicr::WorkItem *d_chunk = nullptr;
    uint64_t chunk_cap = 0;

    // staging of host-resident descriptor tables (returned to `free_stage` at the fence)
    std::vector<hicr::StageBlock> free_stage, used_stage;

    // host threads that check and stage host-resident tables (up to kStageThreadsMax, the caller included)
    hicr::StagePool *stage_pool = nullptr;
    std::atomic<uint64_t> *stage_done = nullptr;
    uint64_t stage_done_cap = 0;

    // counter read-back (pinned): the whole table, for fences the pushed snapshot does not serve
    hicr::SlotCnt *h_fence = nullptr;

    // host-call channel results (mapped pinned)
    hicr::CallResult *h_call = nullptr;
    hicr::CallResult *d_call = nullptr;      // device alias of h_call
    uint64_t call_seq = 0;                   // sequence number of the last host-call push / pop

    // Global Memory Slots (hicr_global.cu).  d_gcnt: owner-side totals of this context's
    // own slots -- every instance that names a global slot adds to them through d_gptr, which holds, per
    // table row of kind GLOBAL, the (possibly peer-mapped) address of the owner's d_gcnt entry.  d_gdelta:
    // what the running batch counted per global row, published to the owner by the batch's last CTA.
    uint32_t instance = 0, n_instances = 1;
    hicr::SlotCnt *d_gcnt = nullptr;         // [HICR_MAX_SLOTS]
    uint64_t *d_gptr = nullptr;              // [HICR_MAX_SLOTS] 0 = not a global row
    hicr::SlotCnt *d_gdelta = nullptr;       // [HICR_MAX_SLOTS] all-zero between batches
    uint32_t n_global = 0;                   // live rows of kind GLOBAL
    hicr::GlobalTable *globals = nullptr;

    // stream capture of a chain of batches (hicr_graph_*)
    bool capturing = false;
    uint32_t captured_batches = 0;
    uint64_t table_version = 0;              // bumped by every change of the slot table
    uint64_t queue_version = 0;              // bumped whenever the chunk queue is re-allocated

    void *launch_cache = nullptr;            // hicr_copy.cu: instantiated one-kernel graphs of recent engine launches

    uint64_t launches = 0;
    int engine_grid = 0;                     // co-resident CTAs of the engine kernel (cooperative launch)
    uint32_t tma_min = hicr::kTmaMinDefault; // HICR_TMA_MIN environment override (0xffffffff = bulk path off)

    bool profiling = false;
    cudaEvent_t ev[2] = {nullptr, nullptr};
    bool ev_valid = false;
    uint64_t last_t[3] = {0, 0, 0};          // %globaltimer stamps of the last completed batch (profile_read)
    uint64_t rec_bad[hicr::kRecRing] = {};   // bad_inv words of the epoch's records, as read at the drain
    std::vector<uint32_t> push_words = std::vector<uint32_t>(hicr::kPushWordsPerSlot * hicr::kPushSlots);
};

namespace hicr {
int cuda_fail(hicr_ctx *ctx, cudaError_t e, const char *what);
int drain_epoch(hicr_ctx *ctx, bool final_fence);
int refresh_counters(hicr_ctx *ctx);
int engine_setup(hicr_ctx *ctx);
void launch_cache_free(hicr_ctx *ctx);
bool table_read_in_place(const hicr_desc_t *descs, uint64_t n);
int stage_table(hicr_ctx *ctx, const hicr_desc_t *descs, uint64_t n, const StageBlock &b, uint64_t *first_bad,
                int *bad_status, uint64_t *n_chunk_bound, uint64_t *n_small, uint64_t *small_bytes);
int bad_to_status(unsigned id);
int slot_install(hicr_ctx *ctx, uint64_t base, uint64_t size, uint64_t flags, hicr_slot_t *out);
int global_setup(hicr_ctx *ctx);
void global_teardown(hicr_ctx *ctx);
int global_forget(hicr_ctx *ctx, uint32_t index);
int pipe_run(hicr_ctx *ctx, const PipeRing *h_rings, PipeRing *d_rings, uint32_t P, uint64_t T, uint64_t C, uint64_t tokens,
             const uint64_t *d_batches, uint64_t n_batches, uint64_t max_batch, CallResult *res, bool *ran);
StagePool *stage_pool_create(int helpers);
void stage_pool_destroy(StagePool *p);
void stage_done_free(std::atomic<uint64_t> *p);

// Table index of a live slot id, or -1 (unknown index, unregistered, or an id from an earlier
// registration of the index).
inline int64_t slot_find(const hicr_ctx *ctx, hicr_slot_t id)
{
    const uint32_t i = id & kSlotIndexMask;
    if (i >= ctx->rows.size()) return -1;
    const SlotRow &r = ctx->rows[i];
    if (r.meta == kInvalidMeta || row_gen(r) != (id >> kSlotIndexBits)) return -1;
    return (int64_t)i;
}
}  // namespace hicr

#define HICR_CUDA(ctx, call)                                                   \
    do {                                                                       \
        cudaError_t e__ = (call);                                              \
        if (e__ != cudaSuccess) return hicr::cuda_fail((ctx), e__, #call);     \
    } while (0)
