// hicr_internal.cuh -- shared declarations of the sm_100a copy engine (not installed).
//
// Layout of the device-side state, the work-item formats produced by the binning
// kernel, and the one copy routine (copy_span) every data-moving kernel uses.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/hicr.h"

namespace hicr {

// ---------------------------------------------------------------- tunables / classes
// size <= kSmallMax  : warp-per-descriptor queue (a4)
// size >  kSmallMax  : split into chunks of kChunkBytes, CTA-per-chunk queue (a5)
constexpr uint64_t kSmallMax = 8192;
constexpr uint64_t kChunkBytes = 32768;
constexpr int kPlanThreads = 256;
constexpr int kCopyThreads = 256;          // 8 warps per CTA in both copy kernels
constexpr int kUnroll = 8;                 // 16-byte vectors in flight per lane
constexpr int kCtlRing = 64;               // control blocks (= batches) per epoch before an internal drain
constexpr uint32_t kSmemSlotHist = 1024;   // per-CTA shared-memory counter histogram up to this many slots

// error ids packed into Ctl::bad (lower id does not mean higher priority; index decides)
constexpr unsigned kBadInvalidSlot = 1, kBadOutOfBounds = 2, kBadNoCapacity = 3;

// One row of the device slot table: "minimum information required to describe a segment
// of memory (e.g., size, starting address)".
struct SlotRow {
    uint64_t base;
    uint64_t size;   // kInvalidSize = not registered
};
constexpr uint64_t kInvalidSize = ~0ull;

// Work item of both copy queues (32 B so that one lane fetches it with two 16 B loads).
struct __align__(16) WorkItem {
    uint64_t src;
    uint64_t dst;
    uint64_t size;
    uint64_t pad;
};

// Per-batch control block, reset to all-zero by one memset at the fence.
struct __align__(64) Ctl {
    unsigned long long bad_inv;  // atomicMax of ~((index << 4) | error id); 0 = no error
    unsigned int n_small;        // items in the warp queue
    unsigned int n_chunk;        // items in the CTA queue
    unsigned int done;           // plan-kernel CTA ticket
    unsigned int go;             // 1 = validated and committed: copy kernels may run
    unsigned int pad[10];
};
static_assert(sizeof(Ctl) == 64, "Ctl is one 64-byte block");

// Channel state in device memory; head and tail on separate 128 B lines so the
// producer's and the consumer's polls do not share a line.
struct __align__(128) ChannelState {
    unsigned long long head;     // tokens ever pushed (producer-advanced)
    unsigned long long pad0[15];
    unsigned long long tail;     // tokens ever popped (consumer-advanced)
    unsigned long long pad1[15];
};
static_assert(sizeof(ChannelState) == 256, "ChannelState is two lines");

// Result of one host-call push/pop, written by the kernel into mapped pinned memory.
struct CallResult {
    unsigned long long k, head, tail;
    long long status;
};

#ifdef __CUDACC__
// ---------------------------------------------------------------- device helpers
enum LdPolicy { kLdStream = 0, kLdL2 = 1 };

template <int POL>
__device__ __forceinline__ uint4 ld16(const uint4 *p)
{
    return POL == kLdStream ? __ldcs(p) : __ldcg(p);
}
template <int POL>
__device__ __forceinline__ unsigned char ld1(const unsigned char *p)
{
    return POL == kLdStream ? __ldcs(p) : __ldcg(p);
}
template <int POL>
__device__ __forceinline__ void st16(uint4 *p, uint4 v)
{
    if (POL == kLdStream) __stcs(p, v); else __stcg(p, v);
}

// dst vector = 16 bytes starting `shift` = 4*Q + r bytes into the 32-byte pair (a, nx).
template <int Q>
__device__ __forceinline__ uint4 shift_combine(const uint4 &a, const uint4 &nx, unsigned rbits)
{
    const unsigned w[8] = {a.x, a.y, a.z, a.w, nx.x, nx.y, nx.z, nx.w};
    uint4 o;
    o.x = __funnelshift_r(w[Q + 0], w[Q + 1], rbits);
    o.y = __funnelshift_r(w[Q + 1], w[Q + 2], rbits);
    o.z = __funnelshift_r(w[Q + 2], w[Q + 3], rbits);
    o.w = __funnelshift_r(w[Q + 3], w[Q + 4], rbits);
    return o;
}

// Body of a copy whose destination is 16 B-aligned and whose source is `4*Q + r` bytes
// past a 16 B boundary (not both zero).  sA = source rounded down to 16 B.  Each warp
// takes tiles of 32*U consecutive destination vectors; lane l loads aligned source
// vectors l, l+32, ... once, and gets the vector after its own from lane l+1 by shuffle
// (lane 31 from lane 0's next load), so every source byte is requested from L2 once.
template <int U, int POL, int Q>
__device__ __forceinline__ void copy_body_shifted(uint4 *__restrict__ d4, const uint4 *__restrict__ sA,
                                                  uint64_t nvec, unsigned rbits, int lane, int warp, int nwarps)
{
    constexpr uint64_t kTile = 32ull * U;
    const uint64_t nfull = nvec / kTile;
    const int nxt_lane = (lane + 1) & 31;
    for (uint64_t t = warp; t < nfull; t += nwarps) {
        const uint64_t base = t * kTile + lane;
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
            st16<POL>(d4 + base + 32 * u, shift_combine<Q>(a[u], nx, rbits));
        }
    }
    const uint64_t rem0 = nfull * kTile;
    if (rem0 < nvec && warp == (int)(nfull % (uint64_t)nwarps)) {
        // ragged last tile: vector v is stored if v < nvec; aligned source vector v is
        // loaded if v <= nvec (vector nvec still holds bytes of destination vector nvec-1)
        const uint64_t base = rem0 + lane;
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
            if (base + 32 * u < nvec) st16<POL>(d4 + base + 32 * u, shift_combine<Q>(a[u], nx, rbits));
        }
    }
}

template <int U, int POL>
__device__ __forceinline__ void copy_body_aligned(uint4 *__restrict__ d4, const uint4 *__restrict__ s4,
                                                  uint64_t nvec, int lane, int warp, int nwarps)
{
    constexpr uint64_t kTile = 32ull * U;
    const uint64_t nfull = nvec / kTile;
    for (uint64_t t = warp; t < nfull; t += nwarps) {
        const uint64_t base = t * kTile + lane;
        uint4 a[U];
#pragma unroll
        for (int u = 0; u < U; u++) a[u] = ld16<POL>(s4 + base + 32 * u);
#pragma unroll
        for (int u = 0; u < U; u++) st16<POL>(d4 + base + 32 * u, a[u]);
    }
    const uint64_t rem0 = nfull * kTile;
    if (rem0 < nvec && warp == (int)(nfull % (uint64_t)nwarps)) {
        const uint64_t base = rem0 + lane;
        uint4 a[U];
#pragma unroll
        for (int u = 0; u < U; u++)
            if (base + 32 * u < nvec) a[u] = ld16<POL>(s4 + base + 32 * u);
#pragma unroll
        for (int u = 0; u < U; u++)
            if (base + 32 * u < nvec) st16<POL>(d4 + base + 32 * u, a[u]);
    }
}

// dst[i] = src[i], i < n, for any alignment of dst and src.  Called by ALL threads of a
// group of `gsize` threads (a multiple of 32: one warp, or a whole CTA), gtid in
// [0, gsize).  Byte head up to the first 16 B boundary of dst, 16 B vector body with
// aligned stores (aligned or byte-shifted loads), byte tail (a4/a5 of SURVEY.md S8(a)).
template <int U, int POL>
__device__ __forceinline__ void copy_span(unsigned char *__restrict__ dst, const unsigned char *__restrict__ src,
                                          uint64_t n, int gtid, int gsize)
{
    const int lane = gtid & 31, warp = gtid >> 5, nwarps = gsize >> 5;
    uint64_t head = (16 - (reinterpret_cast<uintptr_t>(dst) & 15)) & 15;
    if (head > n) head = n;
    if ((uint64_t)gtid < head) dst[gtid] = ld1<POL>(src + gtid);
    dst += head;
    src += head;
    n -= head;
    const uint64_t nvec = n >> 4;
    const unsigned tail = (unsigned)(n & 15);
    {
        const unsigned t = (unsigned)(gsize - 1 - gtid);   // the last threads take the tail
        if (t < tail) dst[nvec * 16 + t] = ld1<POL>(src + nvec * 16 + t);
    }
    if (nvec == 0) return;
    uint4 *d4 = reinterpret_cast<uint4 *>(dst);
    const unsigned s = (unsigned)(reinterpret_cast<uintptr_t>(src) & 15);
    if (s == 0) {
        copy_body_aligned<U, POL>(d4, reinterpret_cast<const uint4 *>(src), nvec, lane, warp, nwarps);
        return;
    }
    const uint4 *sA = reinterpret_cast<const uint4 *>(src - s);
    const unsigned rbits = (s & 3) * 8;
    switch (s >> 2) {
    case 0: copy_body_shifted<U, POL, 0>(d4, sA, nvec, rbits, lane, warp, nwarps); break;
    case 1: copy_body_shifted<U, POL, 1>(d4, sA, nvec, rbits, lane, warp, nwarps); break;
    case 2: copy_body_shifted<U, POL, 2>(d4, sA, nvec, rbits, lane, warp, nwarps); break;
    default: copy_body_shifted<U, POL, 3>(d4, sA, nvec, rbits, lane, warp, nwarps); break;
    }
}

__device__ __forceinline__ unsigned long long ld_acquire(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
#endif  // __CUDACC__

// ---------------------------------------------------------------- host-side context
struct StageBlock {
    void *host = nullptr;   // pinned
    void *dev = nullptr;
    size_t bytes = 0;
};

}  // namespace hicr

struct hicr_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 0;
    std::string cuda_error;

    // slot table: host mirror + device copy
    std::vector<hicr::SlotRow> slots;        // size = ids handed out so far
    std::vector<uint64_t> sent, recv;        // host mirror, refreshed at fence / channel calls
    std::vector<uint32_t> ring_refs;         // live channels using the slot as ring
    hicr::SlotRow *d_slots = nullptr;        // [HICR_MAX_SLOTS]
    unsigned long long *d_sent = nullptr;    // [HICR_MAX_SLOTS]
    unsigned long long *d_recv = nullptr;    // [HICR_MAX_SLOTS]
    unsigned int *d_pending = nullptr;       // [2 * HICR_MAX_SLOTS] per-batch counts before commit
    uint64_t registered_bytes = 0;

    // per-batch control blocks of the current epoch
    hicr::Ctl *d_ctl = nullptr;              // [kCtlRing]
    uint32_t batches_in_epoch = 0;           // since the last fence (or internal drain)
    uint64_t epoch_batch_base = 0;           // batches drained earlier in this epoch
    bool epoch_open = false;                 // any work enqueued since the last fence
    int epoch_error = HICR_OK;               // first deferred error found so far in this epoch
    uint64_t epoch_error_batch = 0, epoch_error_index = 0;
    int last_error = HICR_OK;                // of the last fence, for hicr_fence_error
    uint64_t last_error_batch = 0, last_error_index = 0;

    // work queues
    hicr::WorkItem *d_small = nullptr;
    uint64_t small_cap = 0;
    hicr::WorkItem *d_chunk = nullptr;
    uint64_t chunk_cap = 0;

    // staging of host-resident descriptor tables (returned to `free_stage` at the fence)
    std::vector<hicr::StageBlock> free_stage, used_stage;

    // fence read-back (pinned)
    unsigned char *h_fence = nullptr;
    size_t h_fence_bytes = 0;

    // host-call channel results (mapped pinned)
    hicr::CallResult *h_call = nullptr;
    hicr::CallResult *d_call = nullptr;      // device alias of h_call

    uint64_t launches = 0;
    int copy_ctas_per_sm = 0;

    bool profiling = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool ev_valid = false;
};

namespace hicr {
int cuda_fail(hicr_ctx *ctx, cudaError_t e, const char *what);
int drain_epoch(hicr_ctx *ctx, bool final_fence);
int refresh_counters(hicr_ctx *ctx);
}  // namespace hicr

#define HICR_CUDA(ctx, call)                                                   \
    do {                                                                       \
        cudaError_t e__ = (call);                                              \
        if (e__ != cudaSuccess) return hicr::cuda_fail((ctx), e__, #call);     \
    } while (0)
