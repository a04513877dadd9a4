// hicr_pipe.cu -- the device-resident channel runs as pipelines of bulk copies (a8, a9, a10).
//
// "Channels operate by exchanging pre-allocated circular buffers ... the producer knows where
// to push the next message, as long as the buffer has not filled up. At that point the producer
// may not send any more messages until the consumer notifies that a message has been consumed."
// (PAPER.md:642).  Non-locking MPSC: "dedicated buffers per producer".
//
// The pipe kernels move `tokens` tokens through each of P rings: source -> ring -> sink.  A ring has
// two ENDS, each one CTA, so the single LOGICAL consumer of the MPSC set is P CTAs, one per ring;
// each ring's tail keeps a single writer and each producer's order is kept (per-producer FIFO).
// Head and tail -- the 64-bit counters of ChannelState -- are all the two ends tell each other.
// pipe_cluster_kernel: the ends of ring r are the CTAs of ONE thread-block cluster -- E producer CTAs
// (ranks 0 .. E-1) and E consumer CTAs (ranks E .. 2E-1); E = 1 for many rings, 2 or 4 for a single
// ring (one SM moves 48 GB/s of payload in and out, no more).  The hardware schedules a cluster's
// CTAs together, so the ends may spin on each other whatever else runs (rings are independent: any
// number of rings runs, a wave of clusters at a time), and every CTA writes its progress into the
// shared memory of every CTA of the other end (distributed shared memory), whose workers wait on
// local words.  pipe_kernel (no clusters, or HICR_PIPE_CLUSTER=0): CTA r < P produces, CTA P + r
// consumes, cooperative launch of 2 P co-resident CTAs, the ends poll the counters in L2.
//
// Inside an end the token stream is cut into PIECES -- at the ends of the pushes (the batch list
// of hicr_channel_stream, or every max_batch tokens) and at every multiple of `piece_tokens`
// tokens (a power of two that divides the capacity, so the wrap is a cut too).  Piece g is moved
// by WORKER warp g mod W, whose lane 0 drives 1-D bulk copies (TMA) through the warp's own two
// shared-memory stages:
//   producer  source -> stage, issued one piece ahead (it needs no room in the ring); when tail
//             shows room: stage -> ring, wait until the write is complete;
//   consumer  when head covers the piece: ring -> stage, wait until it has landed (the ring
//             positions are then free); stage -> sink without waiting.
// Each worker publishes, in shared memory, where its next unfinished piece starts.  Pieces tile
// the stream and a worker finishes its own in order, so every token below the MINIMUM of those
// W values is through: that minimum is the CTA's FRONTIER.  One more warp, the COMMITTER, keeps
// taking the minimum (one value per lane, a warp shuffle reduction) and publishes it: "payload
// first, then the counter".  Head needs a device-scope fence between the bulk writes and the
// publication (without it the other end reads stale ring bytes: measured); it is taken by the
// committer once per publication, or by each worker for its own piece where the ring's lap binds.
// Tail needs none: the ring reads behind it have landed.  With several CTAs per end the other end
// takes the minimum over the E frontiers it was told.  The ring stays in L2; DRAM sees the source
// once and the sink once.
//
// Requires T % 16 == 0 and 16 B-aligned ring, source and sink addresses (bulk copies) and a
// piece of at least kPipeMinPiece bytes; other shapes take the vector-copy kernels of hicr_channel.cu.
#include "hicr_internal.cuh"

#include <algorithm>
#include <cstdlib>

namespace hicr {

constexpr int kPipeStages = 2;            // shared-memory stages per worker warp
constexpr int kPipeMaxWorkers = 24;
constexpr unsigned kPipeMinPiece = 1024;  // bytes; below that the per-piece handshakes cost more than the vector kernels

__device__ __forceinline__ unsigned long long ld_acquire_cta_shared_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.cta.shared::cta.u64 %0, [%1];" : "=l"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_cta_shared_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.release.cta.shared::cta.u64 [%0], %1;" ::"r"(smem_u32(p)), "l"(v) : "memory");
}

// ---- thread-block cluster: the producer CTAs and the consumer CTAs of one ring
__device__ __forceinline__ unsigned cluster_ctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release;\nbarrier.cluster.wait.acquire;" ::: "memory");
}
// Store v to the variable at the same shared-memory offset as `local` in CTA `rank` of the cluster.
__device__ __forceinline__ void st_remote_shared_u64(const unsigned long long *local, unsigned rank, unsigned long long v)
{
    unsigned remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(local)), "r"(rank));
    asm volatile("st.relaxed.cluster.shared::cluster.u64 [%0], %1;" ::"r"(remote), "l"(v) : "memory");
}

// The pieces of one end.  Positions are ABSOLUTE token numbers (a = tokens through the ring since
// it was created; ring position = a mod C).  A piece never crosses the end of a push nor a multiple
// of pt = 2^s; pt divides C, so it never crosses the wrap either.  Push i covers [A, B): its
// pieces are the intervals between consecutive cut points, n = ceil(B / pt) - floor(A / pt) of
// them, so a warp steps over a push it has no piece in with a few instructions and finds its own
// pieces (every W-th of the end's) in closed form -- no warp walks the other warps' pieces.
struct PieceWalk {
    unsigned long long A, end, bi, n_batches, jnext, b_cur, b_nxt;
    const unsigned long long *batches;   // tokens per push, or nullptr: every push b_cur tokens
    unsigned s, W;
};
struct Piece {
    unsigned long long a;      // first token (absolute)
    unsigned len;              // tokens
};

__device__ __forceinline__ void walk_init(PieceWalk &w, unsigned long long count0, unsigned long long tokens, unsigned warp,
                                          unsigned W, unsigned s, const unsigned long long *batches,
                                          unsigned long long n_batches, unsigned long long push_tokens)
{
    w.A = count0;
    w.end = count0 + tokens;
    w.bi = 0;
    w.n_batches = n_batches;
    w.jnext = warp;
    w.batches = batches;
    w.s = s;
    w.W = W;
    w.b_cur = batches ? batches[0] : push_tokens;
    w.b_nxt = batches && n_batches > 1 ? batches[1] : push_tokens;
}

// Next piece of this warp, or false when the run is through.
__device__ __forceinline__ bool walk_next_own(PieceWalk &w, Piece &p)
{
    while (w.A < w.end) {
        const unsigned long long B = min(w.A + w.b_cur, w.end);
        const unsigned long long qA = w.A >> w.s, n = ((B + (1ull << w.s) - 1) >> w.s) - qA;   // 0 for a push of no tokens
        if (w.jnext < n) {
            const unsigned long long lo = max(w.A, (qA + w.jnext) << w.s), hi = min(B, (qA + w.jnext + 1) << w.s);
            p.a = lo;
            p.len = (unsigned)(hi - lo);
            w.jnext += w.W;
            return true;
        }
        w.jnext -= n;
        w.A = B;
        w.bi++;
        w.b_cur = w.b_nxt;   // (the size of the push after that is on its way while this one is walked)
        if (w.batches && w.bi + 1 < w.n_batches) w.b_nxt = __ldg(w.batches + w.bi + 1);
    }
    return false;
}

struct PipeArgs {
    const PipeRing *rings;
    uint32_t P;
    uint32_t piece_shift;                // tokens per piece = 1 << piece_shift
    uint32_t stage_bytes;
    uint32_t workers;
    uint32_t ends;                       // CTAs per end (cluster kernel: a cluster holds 2 * ends CTAs)
    uint32_t fence_in_worker;            // cluster kernel: the producer's workers fence their own pieces
    unsigned long long T, C, tokens, max_batch, n_batches;
    const unsigned long long *batches;
    SlotCnt *cnt;
    CallResult *res;                     // ring 0's head / tail at the end of the run (hicr_channel_stream)
};

// The other end's counter as this CTA knows it: the minimum of what the other end's CTAs have written here.
// HICR_MIRROR_ACQUIRE selects how a worker orders the bulk copies (async proxy) that follow a wait behind its
// observation of the other end's frontier (words written with st.relaxed.cluster after the writer's fence):
//   0  plain volatile polls, nothing at the exit of the wait
//   1  every poll is an ld.acquire.cluster; fence.proxy.async at the exit
//   2  volatile polls; fence.acq_rel.cluster + fence.proxy.async at the exit
//   3  volatile polls; fence.proxy.async at the exit
//   5  volatile polls; at the exit the words are read once more with ld.acquire.cluster, then fence.proxy.async
//   6  as 5 without the proxy fence  (DEFAULT)
// Why 6: the ring bytes are written (bulk store) and read (bulk load) through the async proxy on both sides, so
// no location is touched through two proxies; what the reader needs is the acquire that pairs with the writer's
// fence + relaxed store, once per wait.  Measured on B200 (profiles/r03_mirror_acquire.md), config 5a / 5b:
// 0: 63.5 / 4.22 ms, 6: 66.2 / 4.27, 3: 79.1 / 5.01, 5: 81.2 / 5.05, 1: 79.9 / 5.00, 2: 92.8 / 5.95 -- the proxy
// fence at every wait exit is what costs 18-25 %, the acquire 1-4 %.
#ifndef HICR_MIRROR_ACQUIRE
#define HICR_MIRROR_ACQUIRE 6
#endif
__device__ __forceinline__ unsigned long long mirror_word_acquire(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.cluster.shared::cta.u64 %0, [%1];" : "=l"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long mirror_word(const unsigned long long *p)
{
#if HICR_MIRROR_ACQUIRE == 1
    return mirror_word_acquire(p);
#else
    return *reinterpret_cast<const volatile unsigned long long *>(p);
#endif
}
__device__ __forceinline__ unsigned long long mirror_min(const unsigned long long *mirror, unsigned E)
{
    unsigned long long v = mirror_word(mirror);
    for (unsigned t = 1; t < E; t++) v = min(v, mirror_word(mirror + t));
    return v;
}
// At the exit of a successful wait: returns the frontier to go on with (`seen`, or what the acquire reads saw).
__device__ __forceinline__ unsigned long long mirror_wait_done(const unsigned long long *mirror, unsigned E, unsigned long long seen)
{
#if HICR_MIRROR_ACQUIRE == 2
    asm volatile("fence.acq_rel.cluster;" ::: "memory");
#endif
#if HICR_MIRROR_ACQUIRE == 5 || HICR_MIRROR_ACQUIRE == 6
    seen = mirror_word_acquire(mirror);
    for (unsigned t = 1; t < E; t++) seen = min(seen, mirror_word_acquire(mirror + t));
#endif
#if HICR_MIRROR_ACQUIRE == 1 || HICR_MIRROR_ACQUIRE == 2 || HICR_MIRROR_ACQUIRE == 3 || HICR_MIRROR_ACQUIRE == 5
    fence_proxy_async();
#endif
    (void)mirror;
    (void)E;
    return seen;
}

// CL: the two ends of a ring are the two CTAs of a thread-block cluster and tell each other head / tail
// through distributed shared memory (`mirror` of the other CTA) instead of through polls of the
// counters in L2; the counters in device memory follow with plain stores and are final at kernel end.
template <bool CL>
__device__ __forceinline__ void pipe_body(const PipeArgs &a, unsigned char *dyn_smem, uint64_t *bars, unsigned long long *next_start,
                                          unsigned long long *mirror)
{
    const int lane = threadIdx.x & 31;
    const unsigned warp = threadIdx.x >> 5, W = a.workers;
    // cluster: ranks 0 .. E-1 are the producer end's CTAs, E .. 2E-1 the consumer end's; CTA `e` of an end
    // moves the pieces of its own workers
    const unsigned E = CL ? a.ends : 1u, crank = CL ? cluster_ctarank() : 0u;
    const bool producer = CL ? crank < E : blockIdx.x < a.P;
    const unsigned e = CL ? crank % E : 0u;
    const PipeRing r = a.rings[CL ? blockIdx.x / (2 * E) : producer ? blockIdx.x : blockIdx.x - a.P];
    const unsigned long long T = a.T, C = a.C, run_end = r.count0 + a.tokens;
    ChannelState *st = r.st;
    if (threadIdx.x < 32) next_start[threadIdx.x] = threadIdx.x < W ? r.count0 : ~0ull;
    if (threadIdx.x < 8) mirror[threadIdx.x] = threadIdx.x < E ? r.count0 : ~0ull;
    if (lane == 0 && warp < W) {
        for (int s = 0; s < kPipeStages; s++) mbar_init(&bars[warp * kPipeStages + s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (CL) cluster_sync_all();   // both mirrors hold the start value before either end writes the other's

    if (warp == W) {
        // ---- the committer: head (tail) = the frontier, the minimum over the workers of where their
        // first unfinished piece starts.  A worker's bulk writes are complete before it moves its value
        // (release / acquire at CTA scope), and the store below is a release at device scope.
        unsigned long long *counter = producer ? &st->head : &st->tail;
        unsigned long long published = r.count0;
        while (published < run_end) {
            unsigned long long v = ld_acquire_cta_shared_u64(&next_start[lane]);
#pragma unroll
            for (int d = 16; d; d >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, d));
            v = min(v, run_end);          // this CTA's frontier
            if (v > published) {
                if (lane == 0) {
                    // head: payload first, then the counter -- a device-scope fence between them (without it the
                    // consumers read stale ring bytes: measured, 148 rings).  tail: the ring reads behind it have
                    // returned their data (the workers waited on their mbarriers), so plain stores cannot let the
                    // producer overwrite anything still to be read (a second release measured 8 % slower).
                    if (CL) {
                        // every CTA of an end fences its own SM's writes and tells EVERY CTA of the other end its
                        // own frontier (slot e of their `mirror`); they take the minimum themselves
                        if (producer && !a.fence_in_worker) __threadfence();
                        for (unsigned t = 0; t < E; t++) st_remote_shared_u64(&mirror[e], (producer ? E : 0u) + t, v);
                        if (E == 1) *reinterpret_cast<volatile unsigned long long *>(counter) = v;
                    } else if (producer) st_release(counter, v);
                    else *reinterpret_cast<volatile unsigned long long *>(counter) = v;
                }
                published = v;
            }
        }
        // (several CTAs per end: the counter in device memory gets the end's final value; nobody reads it before)
        if (CL && E > 1 && e == 0 && lane == 0) *reinterpret_cast<volatile unsigned long long *>(counter) = run_end;
        if (!producer && e == 0 && lane == 0) {
            // the ring is through: one message per token on every slot it touched (reading 15)
            atomicAdd(&a.cnt[r.id_src].sent, a.tokens);
            atomicAdd(&a.cnt[r.id_ring].recv, a.tokens);
            atomicAdd(&a.cnt[r.id_ring].sent, a.tokens);
            atomicAdd(&a.cnt[r.id_dst].recv, a.tokens);
            if (a.res && blockIdx.x == (CL ? E : a.P)) {
                a.res->k = a.tokens;
                a.res->head = CL ? run_end : ld_acquire(&st->head);
                a.res->tail = published;
                a.res->status = HICR_OK;
                __threadfence_system();
            }
        }
        return;
    }
    if (lane != 0) return;   // one driver lane per worker warp: everything below is bulk-copy issue and waiting

    unsigned char *stage = dyn_smem + (size_t)warp * kPipeStages * a.stage_bytes;
    uint64_t *bar = &bars[warp * kPipeStages];
    PieceWalk wk;
    // the consumer pops what is there: one "push" of all the tokens, no push ends to respect
    walk_init(wk, r.count0, a.tokens, e * W + warp, E * W, a.piece_shift, producer ? a.batches : nullptr,
              producer ? a.n_batches : 0, producer ? a.max_batch : a.tokens);
    const unsigned long long bias = r.count0;     // token a comes from / goes to (a - count0) * T of the source / sink
    unsigned k = 0;   // own pieces so far: stage k % 2, mbarrier parity (k / 2) & 1

    if (producer) {
        Piece cur, nxt;
        bool have = walk_next_own(wk, cur);
        // (until here the worker held the frontier at the start of the run: safe, but the ends would wait
        // for each other for ever if a ring held fewer pieces than an end has workers)
        st_release_cta_shared_u64(&next_start[warp], have ? cur.a : ~0ull);
        if (have) {
            mbar_expect_tx(bar, (unsigned)(cur.len * T));
            bulk_g2s(stage, r.src + (cur.a - bias) * T, (unsigned)(cur.len * T), bar);
        }
        unsigned long long tail_seen = r.count0;   // tail only grows: a stale value is a safe bound
        while (have) {
            const unsigned s = k % kPipeStages, sn = (k + 1) % kPipeStages;
            const bool have_next = walk_next_own(wk, nxt);
            if (have_next) {
                // the other stage is free: the store that last read it was waited for to completion
                mbar_expect_tx(bar + sn, (unsigned)(nxt.len * T));
                bulk_g2s(stage + (size_t)sn * a.stage_bytes, r.src + (nxt.a - bias) * T, (unsigned)(nxt.len * T), bar + sn);
            }
            // room: every position of the piece has been popped ("as long as the buffer has not filled up")
            const unsigned long long end_abs = cur.a + cur.len;
            if (tail_seen + C < end_abs) {
                do tail_seen = CL ? mirror_min(mirror, E) : ld_acquire(&st->tail);
                while (tail_seen + C < end_abs);
                if (CL) tail_seen = mirror_wait_done(mirror, E, tail_seen);
            }
            mbar_wait(bar + s, (k / kPipeStages) & 1);
            bulk_s2g(r.ring + (cur.a % C) * T, stage + (size_t)s * a.stage_bytes, (unsigned)(cur.len * T));
            bulk_commit();
            bulk_wait_all();       // the payload is written (complete, not just read out of shared memory)
            // (where the ring's lap binds -- a single small ring -- the fence head needs is taken here, by every
            // worker for its own piece in parallel, instead of by the committer for all: config 5a 70.6 -> 67.2 ms;
            // where the workers bind -- a large ring -- that costs a quarter of the throughput)
            if (CL && a.fence_in_worker) __threadfence();
            st_release_cta_shared_u64(&next_start[warp], have_next ? nxt.a : ~0ull);   // the committer takes it from here
            cur = nxt;
            have = have_next;
            k++;
        }
        return;
    }

    // ---- consumer worker
    Piece cur;
    unsigned long long head_seen = r.count0;
    bool have = walk_next_own(wk, cur);
    st_release_cta_shared_u64(&next_start[warp], have ? cur.a : ~0ull);
    while (have) {
        const unsigned s = k % kPipeStages;
        const unsigned long long end_abs = cur.a + cur.len;
        if (head_seen < end_abs) {
            do head_seen = CL ? mirror_min(mirror, E) : ld_acquire(&st->head);
            while (head_seen < end_abs);
            if (CL) head_seen = mirror_wait_done(mirror, E, head_seen);
        }
        if (k >= kPipeStages) bulk_wait_read<kPipeStages - 1>();   // the sink store that last read this stage
        const unsigned bytes = (unsigned)(cur.len * T);
        mbar_expect_tx(bar + s, bytes);
        bulk_g2s(stage + (size_t)s * a.stage_bytes, r.ring + (cur.a % C) * T, bytes, bar + s);
        Piece nxt;
        const bool have_next = walk_next_own(wk, nxt);
        mbar_wait(bar + s, (k / kPipeStages) & 1);
        // the ring positions have been read: "the consumer notifies that a message has been consumed"
        // (the wait on the mbarrier is an acquire: the reads are done before the value moves)
        st_release_cta_shared_u64(&next_start[warp], have_next ? nxt.a : ~0ull);
        bulk_s2g(r.dst + (cur.a - bias) * T, stage + (size_t)s * a.stage_bytes, bytes);
        bulk_commit();
        cur = nxt;
        have = have_next;
        k++;
    }
    bulk_wait_all();   // this warp's part of the sink is complete before the CTA may exit
}

__global__ void __launch_bounds__((kPipeMaxWorkers + 1) * 32, 1) pipe_kernel(const PipeArgs a)
{
    extern __shared__ __align__(128) unsigned char dyn_smem[];   // [worker][stage][stage_bytes]
    __shared__ uint64_t bars[kPipeMaxWorkers * kPipeStages];
    __shared__ unsigned long long next_start[32];                // per worker: first token of its first unfinished piece
    __shared__ unsigned long long mirror[8];
    pipe_body<false>(a, dyn_smem, bars, next_start, mirror);
}

__global__ void __launch_bounds__((kPipeMaxWorkers + 1) * 32, 1) pipe_cluster_kernel(const PipeArgs a)
{
    extern __shared__ __align__(128) unsigned char dyn_smem[];
    __shared__ uint64_t bars[kPipeMaxWorkers * kPipeStages];
    __shared__ unsigned long long next_start[32];
    __shared__ unsigned long long mirror[8];                     // slot e: the frontier of CTA e of the other end, written by it
    pipe_body<true>(a, dyn_smem, bars, next_start, mirror);
    cluster_sync_all();   // neither CTA leaves while the other may still write its mirror
}

// Shape of a run: workers per end, stage size, tokens per piece; false if the bulk-copy pipeline
// cannot take it (alignment, pieces too small).  coresident: all 2 P CTAs fit the device at once, which the
// cooperative variant needs (its ends spin on each other across CTAs the hardware schedules one by one);
// the cluster variant does not: a ring's two ends are one cluster, scheduled together, and rings are
// independent, so any number of rings runs, a wave of clusters at a time.
struct PipeShape {
    unsigned workers, stage_bytes, piece_shift;
    size_t smem;
    bool coresident;
};

static bool pipe_shape(hicr_ctx *ctx, uint32_t P, uint64_t T, uint64_t C, PipeShape *out)
{
    if (T % 16 != 0 || T == 0) return false;
    int max_smem = 0;
    if (cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device) != cudaSuccess) return false;
    // CTAs that share an SM (at most two: beyond that the rings run in waves)
    const unsigned per_sm = std::min<unsigned>(2u, (2 * P + ctx->num_sms - 1) / ctx->num_sms);
    // shared memory of an SM, less what the system keeps per CTA and the static part
    const size_t budget = std::min<size_t>((size_t)max_smem, (size_t)(228 * 1024) / per_sm - 2048);
    // Per CTA: 6 workers x 2 stages x 16 KiB for one ring (config 5a: 63.7 ms against 67.3 with 12 x 8 KiB, 73.3
    // with 24 x 4 KiB), 3 x 2 x 16 KiB for many rings, two CTAs per SM (148 rings: 4.23 ms against 4.33 with
    // 6 x 8 KiB and 4.57 with 12 x 4 KiB): fewer, larger pieces mean fewer publications per lap.
    unsigned stage = 16384;
    while (stage < T && (size_t)kPipeStages * 2 * stage <= budget) stage *= 2;
    while (stage > 1024 && budget < (size_t)kPipeStages * stage) stage /= 2;
    unsigned workers = (unsigned)std::min<size_t>(budget / ((size_t)kPipeStages * stage), P == 1 ? 6 : 3);
    workers = std::min<unsigned>(workers, kPipeMaxWorkers);
    if (workers < 1) return false;
    // tokens per piece: the largest power of two that divides C and fits a stage (the wrap is then a cut too)
    unsigned shift = 0;
    while (((C >> (shift + 1)) << (shift + 1)) == C && (T << (shift + 1)) <= stage) shift++;
    if (T > stage || (T << shift) < kPipeMinPiece) return false;
    out->workers = workers;
    out->stage_bytes = stage;
    out->piece_shift = shift;
    out->smem = (size_t)workers * kPipeStages * stage;
    if (out->smem > (size_t)max_smem) return false;
    if (cudaFuncSetAttribute(pipe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)out->smem) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    int resident = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, pipe_kernel, (int)(32 * (workers + 1)), out->smem) !=
        cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    out->coresident = (uint64_t)resident * ctx->num_sms >= 2ull * P;
    return true;
}

// Runs the pipeline if the shape allows it (*ran = true) on the context's stream; the caller
// synchronises.  h_rings: P host records; d_rings: device space for them; d_batches: the push
// sizes on the device (n_batches of them), or nullptr for pushes of max_batch tokens.
int pipe_run(hicr_ctx *ctx, const PipeRing *h_rings, PipeRing *d_rings, uint32_t P, uint64_t T, uint64_t C, uint64_t tokens,
             const uint64_t *d_batches, uint64_t n_batches, uint64_t max_batch, CallResult *res, bool *ran)
{
    *ran = false;
    PipeShape sh;
    for (uint32_t p = 0; p < P; p++) {
        const uintptr_t bits = (uintptr_t)h_rings[p].ring | (uintptr_t)h_rings[p].src | (uintptr_t)h_rings[p].dst;
        if (bits % 16) return HICR_OK;
    }
    if (!pipe_shape(ctx, P, T, C, &sh)) return HICR_OK;
    HICR_CUDA(ctx, cudaMemcpyAsync(d_rings, h_rings, sizeof(PipeRing) * P, cudaMemcpyHostToDevice, ctx->stream));
    PipeArgs a;
    a.rings = d_rings;
    a.P = P;
    a.piece_shift = sh.piece_shift;
    a.stage_bytes = sh.stage_bytes;
    a.workers = sh.workers;
    a.ends = 1;
    a.fence_in_worker = 0;
    a.T = T;
    a.C = C;
    a.tokens = tokens;
    a.max_batch = max_batch;
    a.n_batches = n_batches;
    a.batches = reinterpret_cast<const unsigned long long *>(d_batches);
    a.cnt = ctx->d_cnt;
    a.res = res;
    void *args[] = {&a};
    // The two ends of a ring as ONE thread-block cluster: the hardware schedules both CTAs together, so the
    // ends can spin on each other whatever else runs on the device (rings do not depend on one another), and
    // they signal through distributed shared memory (148 rings: 5.2 -> 4.5 ms).  Without cluster support for
    // this shape: a cooperative launch of 2 P separate CTAs, signalling through the counters in L2.
    bool clustered = false;
    // HICR_PIPE_CLUSTER=0 forces the cooperative path (the tests run both; read per call)
    const char *knob = getenv("HICR_PIPE_CLUSTER");
    if (!(knob && knob[0] == '0')) {
        // CTAs per end.  One SM moves about 93 GB/s through its L2 port, i.e. 48 GB/s of payload in and out:
        // a single ring gets two CTAs per end (config 5a: the lap of its 256 KiB ring then binds, 50.8 GB/s),
        // four when the ring is large enough not to (1 MiB: 96 GB/s with two, 156-188 GB/s with four);
        // many rings get one CTA per end and fill the device that way.
        const unsigned E = P > 1 ? 1u : C * T >= (1u << 20) ? 4u : 2u;
        a.ends = E;
        a.fence_in_worker = E == 2 || P > 1;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(2 * E * P);
        cfg.blockDim = dim3(32 * (sh.workers + 1));
        cfg.dynamicSmemBytes = sh.smem;
        cfg.stream = ctx->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = 2 * E;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        int n_clusters = 0;
        cudaError_t e = cudaFuncSetAttribute(pipe_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh.smem);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveClusters(&n_clusters, (const void *)pipe_cluster_kernel, &cfg);
        if (e == cudaSuccess && n_clusters >= 1) {
            e = cudaLaunchKernelExC(&cfg, (const void *)pipe_cluster_kernel, args);
            clustered = e == cudaSuccess;
        }
        if (!clustered) {
            (void)cudaGetLastError();
            a.ends = 1;
            a.fence_in_worker = 0;
        }
    }
    if (!clustered && !sh.coresident) return HICR_OK;   // too many rings for a cooperative launch: the caller's other path
    if (!clustered)
    HICR_CUDA(ctx, cudaLaunchCooperativeKernel((const void *)pipe_kernel, dim3(2 * P), dim3(32 * (sh.workers + 1)), args,
                                               sh.smem, ctx->stream));
    ctx->launches++;
    ctx->push_stale = true;
    *ran = true;
    return HICR_OK;
}

}  // namespace hicr
