// hicr_channel.cu -- fixed-size-token channels on device counters (a8, a9, a10).
//
// "Channels operate by exchanging pre-allocated circular buffers ... By pre-allocating
// the buffers, the producer knows where to push the next message, as long as the buffer
// has not filled up. At that point the producer may not send any more messages until the
// consumer notifies that a message has been consumed.".  MPSC non-locking:
// "dedicated buffers per producer".
//
// head (tokens ever pushed) and tail (tokens ever popped) are 64-bit counters in device
// memory; the push/pop decision k is taken on the device from them.  Payload first, then
// the counter with release semantics; the other side reads the counter with acquire.
//
//   channel_push_kernel / channel_pop_kernel  one call = one launch; the grid splits the
//        (at most two) contiguous spans into pieces; the last CTA to finish publishes the
//        counter, the slot message counts and the call result (mapped pinned memory).
//   spsc_stream_kernel   cooperative launch, CTA 0 = producer, CTA 1 = consumer, the whole
//        push/pop sequence in one kernel (no host round trip per call).
//   mpsc_stream_kernel   cooperative launch, CTA p < P = producer p (one per SM for P = 148),
//        CTA P = the single consumer; its warps each poll and drain their own rings.
#include "hicr_internal.cuh"

#include <algorithm>
#include <cstring>

struct hicr_channel {
    hicr_ctx *ctx = nullptr;
    uint32_t ring = 0;             // table index of the ring slot
    uint64_t T = 0, C = 0;
    hicr::ChannelState *d_state = nullptr;
    unsigned int *d_ticket = nullptr;
    uint64_t head = 0, tail = 0;   // host mirror as of the last completed call
    hicr::NodeLauncher call[2];    // one-kernel graphs of the host-call push (0) and pop (1)
    bool call_plain = false;       // the graph path was refused once
    // device scratch of the device-resident runs, kept between calls (grown on demand)
    unsigned char *d_tab = nullptr;
    size_t tab_bytes = 0;
};

struct hicr_mpsc {
    hicr_ctx *ctx = nullptr;
    uint32_t P = 0;
    uint64_t T = 0, C = 0;
    std::vector<uint32_t> rings;             // table indices of the ring slots
    hicr::ChannelState *d_state = nullptr;   // [P]
    uint64_t *d_ptrs = nullptr;              // [4 * P] u64: ring base, source address, sink address, tokens before the run;
                                             // then [3 * P] u32: table indices of ring, source, sink
    hicr::PipeRing *d_pipe = nullptr;        // [P] ring records of the bulk-copy pipeline (hicr_pipe.cu)
    std::vector<uint64_t> head, tail;
};

namespace hicr {

constexpr int kCallThreads = 256;
constexpr uint64_t kPieceBytes = 16384;     // per-CTA piece of a host-call push/pop
constexpr int kStreamThreads = 512;   // SPSC stream: 2 CTAs on 2 SMs
constexpr int kMpscThreads = 256;     // MPSC stream: P + 1 CTAs must be co-resident, 2 per SM at <= 128 registers

// Copy `len` logical bytes starting at logical ring byte `rb` (wraps at ring_bytes).
template <int U, bool TO_RING>
__device__ __forceinline__ void ring_copy(unsigned char *ring, uint64_t ring_bytes, uint64_t rb,
                                          unsigned char *lin, uint64_t len, int gtid, int gsize)
{
    const uint64_t first = min(len, ring_bytes - rb);
    if (TO_RING) {
        copy_span<U, kLdL2>(ring + rb, lin, first, gtid, gsize);
        if (len > first) copy_span<U, kLdL2>(ring, lin + first, len - first, gtid, gsize);
    } else {
        copy_span<U, kLdL2>(lin, ring + rb, first, gtid, gsize);
        if (len > first) copy_span<U, kLdL2>(lin + first, ring, len - first, gtid, gsize);
    }
}

// (a8) push / (a9) pop as one launch.  `lin` = the linear side (source slot for push,
// destination slot for pop) already offset; lin_room = bytes available there.
template <bool PUSH>
__global__ void __launch_bounds__(kCallThreads)
channel_call_kernel(ChannelState *st, unsigned int *ticket, unsigned char *ring, uint64_t T, uint64_t C,
                    unsigned char *lin, uint64_t lin_room, uint64_t n, unsigned long long *cnt_lin_out,
                    unsigned long long *cnt_ring_out, CallResult *res, unsigned long long seq)
{
    const unsigned long long head = st->head, tail = st->tail;
    uint64_t k;
    long long status = HICR_OK;
    if (PUSH) k = min((unsigned long long)n, (unsigned long long)C - (head - tail));
    else {
        k = min((unsigned long long)n, head - tail);
        if (k * T > lin_room) {   // destination range of the k tokens must fit (no effect otherwise)
            status = HICR_ERR_OUT_OF_BOUNDS;
            k = 0;
        }
    }
    const uint64_t bytes = k * T, ring_bytes = C * T;
    const uint64_t rb0 = ((PUSH ? head : tail) % C) * T;
    for (uint64_t off = (uint64_t)blockIdx.x * kPieceBytes; off < bytes; off += (uint64_t)gridDim.x * kPieceBytes) {
        const uint64_t len = min(kPieceBytes, bytes - off);
        ring_copy<4, PUSH>(ring, ring_bytes, (rb0 + off) % ring_bytes, lin + off, len, threadIdx.x, kCallThreads);
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    // release: this CTA's copies (ordered before it by the barrier); acquire: the other CTAs'
    if (atom_inc_acq_rel_u32(ticket) != gridDim.x - 1) return;
    // last CTA: every CTA has read head/tail and finished its pieces
    *ticket = 0;
    unsigned long long new_head = head, new_tail = tail;
    if (PUSH) {
        new_head = head + k;
        st->head = new_head;
        *cnt_lin_out += k;     // sent(src)
        *cnt_ring_out += k;    // recv(ring)
    } else {
        new_tail = tail + k;
        st->tail = new_tail;
        *cnt_ring_out += k;    // sent(ring)
        *cnt_lin_out += k;     // recv(dst)
    }
    // ONE device-scope fence: payload, counter and message counts are performed before the
    // result leaves for the host.  The result itself is seven flagged 8-byte words (payload
    // low, flag high, as the engine's completion record): a word whose flag matches carries
    // its value, so no system-scope fence is needed (1.6 us each).
    __threadfence();
    const uint32_t flag = rec_flag(seq);
    unsigned long long *w = res->w;
    const unsigned long long vals[3] = {k, new_head, new_tail};
#pragma unroll
    for (int i = 0; i < 3; i++) {
        *reinterpret_cast<volatile unsigned long long *>(w + 2 * i) = ((unsigned long long)flag << 32) | (uint32_t)vals[i];
        *reinterpret_cast<volatile unsigned long long *>(w + 2 * i + 1) = ((unsigned long long)flag << 32) | (uint32_t)(vals[i] >> 32);
    }
    *reinterpret_cast<volatile unsigned long long *>(w + 6) = ((unsigned long long)flag << 32) | (uint32_t)status;
}

__device__ __forceinline__ void backoff(unsigned &ns)
{
    __nanosleep(ns);
    if (ns < 256) ns *= 2;
}

// Device-resident SPSC run.  CTA 0 produces, CTA 1 consumes; co-residency is guaranteed by
// the cooperative launch.  cnt[0..3] = &sent[src], &recv[ring], &sent[ring], &recv[dst].
__global__ void __launch_bounds__(kStreamThreads)
spsc_stream_kernel(ChannelState *st, unsigned char *ring, uint64_t T, uint64_t C, unsigned char *src,
                   unsigned char *dst, const uint64_t *__restrict__ batches, uint64_t n_batches, uint64_t total,
                   unsigned long long *c_sent_src, unsigned long long *c_recv_ring,
                   unsigned long long *c_sent_ring, unsigned long long *c_recv_dst, CallResult *res)
{
    __shared__ unsigned long long sh_k;
    const uint64_t ring_bytes = C * T;
    const int tid = threadIdx.x;
    if (blockIdx.x == 0) {
        unsigned long long head = st->head, tail_seen = st->tail;   // tail only grows: a stale value is a safe bound
        uint64_t pushed = 0;
        for (uint64_t b = 0; b < n_batches; b++) {
            uint64_t rem = batches[b];
            while (rem) {            // blocking push: wait for room, push what fits
                if (tid == 0) {
                    unsigned long long room = C - (head - tail_seen);
                    if (room < rem) {   // look at the consumer's counter only when the known room is short
                        unsigned ns = 20;
                        while ((room = C - (head - (tail_seen = ld_acquire(&st->tail)))) == 0) backoff(ns);
                    }
                    sh_k = min((unsigned long long)rem, room);
                }
                __syncthreads();
                const uint64_t k = sh_k;
                ring_copy<8, true>(ring, ring_bytes, (head % C) * T, src + pushed * T, k * T, tid, kStreamThreads);
                __syncthreads();     // every thread's payload stores are issued
                // payload before counter: the release covers the CTA's stores ordered before it by the barrier
                if (tid == 0) st_release(&st->head, head + k);
                head += k;
                pushed += k;
                rem -= k;
            }
        }
    } else {
        unsigned long long tail = st->tail;
        uint64_t popped = 0;
        while (popped < total) {
            if (tid == 0) {
                unsigned ns = 20;
                unsigned long long avail;
                while ((avail = ld_acquire(&st->head) - tail) == 0) backoff(ns);
                sh_k = avail;
            }
            __syncthreads();
            const uint64_t k = sh_k;
            ring_copy<8, false>(ring, ring_bytes, (tail % C) * T, dst + popped * T, k * T, tid, kStreamThreads);
            __syncthreads();         // every thread's ring loads have returned (their stores were issued)
            if (tid == 0) st_release(&st->tail, tail + k);
            tail += k;
            popped += k;
        }
        if (tid == 0) {
            atomicAdd(c_sent_src, total);
            atomicAdd(c_recv_ring, total);
            atomicAdd(c_sent_ring, total);
            atomicAdd(c_recv_dst, total);
            res->k = total;
            res->head = ld_acquire(&st->head);
            res->tail = tail;
            res->status = HICR_OK;
            __threadfence_system();
        }
    }
}

// Device-resident non-locking MPSC run.  ptrs = [ring base | source address | sink address | tokens
// through the ring before this run] x P; slot_ids = [ring | source | sink] x P (table indices) for
// the message counters.  head/tail keep counting from where the last run (or call) left them.
__global__ void __launch_bounds__(kMpscThreads, 2)
mpsc_stream_kernel(ChannelState *st, uint32_t P, uint64_t T, uint64_t C, const uint64_t *__restrict__ ptrs,
                   const uint32_t *__restrict__ slot_ids, uint64_t tokens, uint64_t max_batch, SlotCnt *cnt)
{
    const uint64_t ring_bytes = C * T;
    const int tid = threadIdx.x;
    if (blockIdx.x < P) {
        // ---- producer p: blocking pushes of at most max_batch tokens
        __shared__ unsigned long long sh_k;
        const uint32_t p = blockIdx.x;
        ChannelState *s = st + p;
        unsigned char *ring = reinterpret_cast<unsigned char *>(ptrs[p]);
        unsigned char *src = reinterpret_cast<unsigned char *>(ptrs[P + p]);
        unsigned long long head = s->head;
        uint64_t pushed = 0;
        while (pushed < tokens) {
            if (tid == 0) {
                unsigned ns = 20;
                unsigned long long room;
                while ((room = C - (head - ld_acquire(&s->tail))) == 0) backoff(ns);
                sh_k = min(min((unsigned long long)(tokens - pushed), (unsigned long long)max_batch), room);
            }
            __syncthreads();
            const uint64_t k = sh_k;
            ring_copy<2, true>(ring, ring_bytes, (head % C) * T, src + pushed * T, k * T, tid, kMpscThreads);
            __syncthreads();
            if (tid == 0) st_release(&s->head, head + k);
            head += k;
            pushed += k;
        }
        return;
    }
    // ---- the single consumer: warp w polls and drains rings w, w + nwarps, ...
    const int lane = tid & 31, warp = tid >> 5, nwarps = kMpscThreads / 32;
    bool all_done = false;
    unsigned ns = 20;
    while (!all_done) {
        all_done = true;
        bool progressed = false;
        for (uint32_t p = warp; p < P; p += nwarps) {
            ChannelState *s = st + p;
            unsigned long long tail = 0, head = 0;
            const unsigned long long end = ptrs[3 * P + p] + tokens;   // tail when this run is through
            if (lane == 0) {
                tail = __ldcg(&s->tail);   // only this warp ever writes it (read at L2, where the release store went)
                head = tail < end ? ld_acquire(&s->head) : tail;
            }
            tail = __shfl_sync(0xffffffffu, tail, 0);
            head = __shfl_sync(0xffffffffu, head, 0);
            if (tail >= end) continue;
            all_done = false;
            const uint64_t k = head - tail;
            if (k == 0) continue;
            progressed = true;
            unsigned char *ring = reinterpret_cast<unsigned char *>(ptrs[p]);
            // sink address of the token at ring count `tail`
            unsigned char *dst = reinterpret_cast<unsigned char *>(ptrs[2 * P + p]) - (end - tokens) * T;
            ring_copy<4, false>(ring, ring_bytes, (tail % C) * T, dst + tail * T, k * T, lane, 32);
            __syncwarp();
            if (lane == 0) {
                st_release(&s->tail, tail + k);
                if (tail + k == end) {   // this ring is through: one message per token (reading 15)
                    atomicAdd(&cnt[slot_ids[P + p]].sent, (unsigned long long)tokens);
                    atomicAdd(&cnt[slot_ids[p]].recv, (unsigned long long)tokens);
                    atomicAdd(&cnt[slot_ids[p]].sent, (unsigned long long)tokens);
                    atomicAdd(&cnt[slot_ids[2 * P + p]].recv, (unsigned long long)tokens);
                }
            }
        }
        if (!progressed && !all_done) backoff(ns); else ns = 20;
    }
}

// Device-resident LOCKING MPSC run ("locking, where a collective exclusive access
// guarantees a shared channel does not overflow"): P producer CTAs share ONE ring.  The
// exclusive access is an atomic reservation: a producer advances `reserve` by k only if the k
// positions are free (reserve + k - tail <= C, compare-and-swap), copies its tokens into the
// positions it owns, and commits in reservation order -- it waits until head has reached its
// first position and then moves head past its last one.  Each wait is on a producer that
// reserved earlier and is co-resident (cooperative launch), so the chain always advances.
// CTA P is the single consumer: pops whatever head shows into dst, consecutively.
// srcs = source base addresses x P; slot_ids = source slot ids x P (message counters).
__global__ void __launch_bounds__(kMpscThreads, 2)
mpsc_locking_kernel(ChannelState *st, unsigned long long *reserve, uint32_t P, unsigned char *ring, uint64_t T,
                    uint64_t C, const uint64_t *__restrict__ srcs, const uint32_t *__restrict__ slot_ids,
                    unsigned char *dst, uint64_t tokens, uint64_t max_batch, SlotCnt *cnt, uint32_t ring_slot,
                    uint32_t dst_slot, CallResult *res)
{
    __shared__ unsigned long long sh_start, sh_k;
    const uint64_t ring_bytes = C * T;
    const int tid = threadIdx.x;
    if (blockIdx.x < P) {
        const uint32_t p = blockIdx.x;
        unsigned char *src = reinterpret_cast<unsigned char *>(srcs[p]);
        uint64_t pushed = 0;
        while (pushed < tokens) {
            if (tid == 0) {
                const unsigned long long want = min((unsigned long long)(tokens - pushed), (unsigned long long)max_batch);
                unsigned ns = 20;
                for (;;) {
                    const unsigned long long r = *reinterpret_cast<volatile unsigned long long *>(reserve);
                    const unsigned long long room = C - (r - ld_acquire(&st->tail));   // tail <= head <= reserve
                    if (room == 0 || room > C) {   // full (or a tail newer than the reserve value just read)
                        backoff(ns);
                        continue;
                    }
                    const unsigned long long k = min(want, room);
                    if (atomicCAS(reserve, r, r + k) == r) {
                        sh_start = r;
                        sh_k = k;
                        break;
                    }
                }
            }
            __syncthreads();
            const uint64_t start = sh_start, k = sh_k;
            ring_copy<2, true>(ring, ring_bytes, (start % C) * T, src + pushed * T, k * T, tid, kMpscThreads);
            __syncthreads();
            if (tid == 0) {
                while (ld_acquire(&st->head) != start) {}   // commit in reservation order (the wait is on the critical path
                                                            // of the ring's lap: no back-off)
                st_release(&st->head, start + k);
            }
            pushed += k;
        }
        if (tid == 0) atomicAdd(&cnt[slot_ids[p]].sent, (unsigned long long)tokens);
        return;
    }
    // ---- the single consumer
    const uint64_t total = (uint64_t)P * tokens;
    unsigned long long tail = st->tail;
    const unsigned long long tail0 = tail;
    uint64_t popped = 0;
    while (popped < total) {
        if (tid == 0) {
            unsigned ns = 20;
            unsigned long long avail;
            while ((avail = ld_acquire(&st->head) - tail) == 0) backoff(ns);
            sh_k = avail;
        }
        __syncthreads();
        const uint64_t k = sh_k;
        ring_copy<4, false>(ring, ring_bytes, (tail % C) * T, dst + popped * T, k * T, tid, kMpscThreads);
        __syncthreads();
        // (every thread's ring loads have returned -- their values went into the stores before the barrier -- so a
        // plain store frees the positions; a release would also wait for the sink stores to drain)
        if (tid == 0) *reinterpret_cast<volatile unsigned long long *>(&st->tail) = tail + k;
        tail += k;
        popped += k;
    }
    if (tid == 0) {
        atomicAdd(&cnt[ring_slot].recv, (unsigned long long)total);
        atomicAdd(&cnt[ring_slot].sent, (unsigned long long)total);
        atomicAdd(&cnt[dst_slot].recv, (unsigned long long)total);
        res->k = total;
        res->head = tail0 + total;
        res->tail = tail;
        res->status = HICR_OK;
        __threadfence_system();
    }
}

// The kernel wrote the result into mapped pinned memory before the stream synchronize returned.
static CallResult read_result(hicr_ctx *ctx)
{
    const volatile CallResult *v = ctx->h_call;
    CallResult r;
    r.k = v->k;
    r.head = v->head;
    r.tail = v->tail;
    r.status = v->status;
    return r;
}

// Device scratch of a channel's device-resident runs: at least `bytes`, contents undefined.
static int channel_scratch(hicr_channel *ch, size_t bytes)
{
    if (bytes <= ch->tab_bytes) return HICR_OK;
    hicr_ctx *ctx = ch->ctx;
    HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (ch->d_tab) HICR_CUDA(ctx, cudaFree(ch->d_tab));
    ch->d_tab = nullptr;
    ch->tab_bytes = 0;
    const size_t cap = std::max<size_t>(bytes, 1 << 16);
    HICR_CUDA(ctx, cudaMalloc(&ch->d_tab, cap));
    ch->tab_bytes = cap;
    return HICR_OK;
}

// Overflow-safe "count tokens of T bytes fit into [off, size)".
static bool tokens_fit(uint64_t count, uint64_t T, uint64_t off, uint64_t size)
{
    return off <= size && (count == 0 || (count <= ~0ull / T && count * T <= size - off));
}

}  // namespace hicr

using namespace hicr;

extern "C" {

int hicr_channel_create(hicr_ctx_t *ctx, hicr_slot_t ring, uint64_t token_bytes, uint64_t capacity,
                        hicr_channel_t **out)
{
    if (!ctx || !out) return HICR_ERR_INVALID_ARG;
    *out = nullptr;
    if (token_bytes == 0 || capacity == 0) return HICR_ERR_INVALID_ARG;   // capacity >= 1
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    const int64_t ri = slot_find(ctx, ring);
    if (ri < 0) return HICR_ERR_INVALID_SLOT;
    if (!tokens_fit(capacity, token_bytes, 0, row_size(ctx->rows[ri]))) return HICR_ERR_OUT_OF_BOUNDS;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    hicr_channel *ch = new hicr_channel();
    ch->ctx = ctx;
    ch->ring = (uint32_t)ri;
    ch->T = token_bytes;
    ch->C = capacity;
    cudaError_t e = cudaMalloc(&ch->d_state, sizeof(ChannelState) + 128);
    if (e == cudaSuccess) e = cudaMemsetAsync(ch->d_state, 0, sizeof(ChannelState) + 128, ctx->stream);
    if (e != cudaSuccess) {
        cudaFree(ch->d_state);
        delete ch;
        return cuda_fail(ctx, e, "hicr_channel_create");
    }
    ch->d_ticket = reinterpret_cast<unsigned int *>(ch->d_state + 1);
    ctx->ring_refs[ri]++;
    *out = ch;
    return HICR_OK;
}

int hicr_channel_destroy(hicr_channel_t *ch)
{
    if (!ch) return HICR_ERR_INVALID_ARG;
    if (ch->ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    (void)cudaStreamSynchronize(ch->ctx->stream);
    cudaFree(ch->d_state);
    cudaFree(ch->d_tab);
    node_free(ch->call[0]);
    node_free(ch->call[1]);
    ch->ctx->ring_refs[ch->ring]--;
    delete ch;
    return HICR_OK;
}

int hicr_channel_counters(hicr_channel_t *ch, uint64_t *head, uint64_t *tail)
{
    if (!ch || !head || !tail) return HICR_ERR_INVALID_ARG;
    *head = ch->head;
    *tail = ch->tail;
    return HICR_OK;
}

static int channel_call(hicr_channel_t *ch, bool push, hicr_slot_t lin_slot, uint64_t off, uint64_t n,
                        uint64_t *n_out)
{
    if (!ch || !n_out) return HICR_ERR_INVALID_ARG;
    hicr_ctx *ctx = ch->ctx;
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    *n_out = 0;
    const int64_t li = slot_find(ctx, lin_slot);
    if (li < 0) return HICR_ERR_INVALID_SLOT;
    const SlotRow &ls = ctx->rows[li];
    const uint64_t lsize = row_size(ls);
    if (off > lsize) return HICR_ERR_OUT_OF_BOUNDS;
    if (push && !tokens_fit(n, ch->T, off, lsize)) return HICR_ERR_OUT_OF_BOUNDS;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    const uint64_t max_tokens = std::min<uint64_t>(n, ch->C);
    const uint64_t max_bytes = max_tokens * ch->T;
    unsigned grid = (unsigned)std::min<uint64_t>(std::max<uint64_t>(1, (max_bytes + kPieceBytes - 1) / kPieceBytes),
                                                 (uint64_t)ctx->num_sms * 4);
    unsigned char *ring = reinterpret_cast<unsigned char *>(ctx->rows[ch->ring].base);
    unsigned char *lin = reinterpret_cast<unsigned char *>(ls.base + off);
    CallResult *res = ctx->d_call;
    const unsigned long long seq = ++ctx->call_seq;
    SlotCnt *cl = ctx->d_cnt + li, *cr = ctx->d_cnt + ch->ring;
    // (one-kernel graph with rewritten parameters: starts sooner than a stream launch, see NodeLauncher)
    bool launched = false;
    if (!ch->call_plain) {
        ChannelState *st = ch->d_state;
        unsigned int *tk = ch->d_ticket;
        uint64_t T = ch->T, C = ch->C, room = lsize - off, nn = n;
        unsigned long long *c_lin = push ? &cl->sent : &cl->recv, *c_ring = push ? &cr->recv : &cr->sent, sq = seq;
        void *args[] = {&st, &tk, &ring, &T, &C, &lin, &room, &nn, &c_lin, &c_ring, &res, &sq};
        const void *fn = push ? (const void *)channel_call_kernel<true> : (const void *)channel_call_kernel<false>;
        launched = node_launch(ch->call[push ? 0 : 1], fn, dim3(grid), dim3(kCallThreads), 0, args, false, true, ctx->stream) ==
                   cudaSuccess;
        if (!launched) ch->call_plain = true;
    }
    if (!launched) {
        if (push)
            channel_call_kernel<true><<<grid, kCallThreads, 0, ctx->stream>>>(
                ch->d_state, ch->d_ticket, ring, ch->T, ch->C, lin, lsize - off, n, &cl->sent, &cr->recv, res, seq);
        else
            channel_call_kernel<false><<<grid, kCallThreads, 0, ctx->stream>>>(
                ch->d_state, ch->d_ticket, ring, ch->T, ch->C, lin, lsize - off, n, &cl->recv, &cr->sent, res, seq);
    }
    ctx->launches++;
    ctx->push_stale = true;   // the device counters moved after the last batch's pushed snapshot
    HICR_CUDA(ctx, cudaGetLastError());
    // "Complete on return": the last CTA writes the result as flagged words, which the host polls
    // (4.5 us less per call than cudaStreamSynchronize); every so often the stream is asked,
    // so a fault is not a hang
    CallResult r;
    {
        const volatile unsigned long long *w = ctx->h_call->w;
        const uint32_t flag = rec_flag(seq);
        unsigned long long v[7];
        unsigned spins = 0;
        for (int i = 0; i < 7; i++) {
            while ((uint32_t)((v[i] = w[i]) >> 32) != flag) {
                if ((++spins & 0x3fff) == 0) {
                    cudaError_t qe = cudaStreamQuery(ctx->stream);
                    if (qe == cudaSuccess) {
                        if ((uint32_t)((v[i] = w[i]) >> 32) == flag) break;
                        ctx->cuda_error = "channel kernel finished without publishing its result";
                        return HICR_ERR_CUDA;
                    }
                    if (qe != cudaErrorNotReady) return cuda_fail(ctx, qe, "cudaStreamQuery(channel call)");
                }
            }
        }
        r.k = (uint32_t)v[0] | ((unsigned long long)(uint32_t)v[1] << 32);
        r.head = (uint32_t)v[2] | ((unsigned long long)(uint32_t)v[3] << 32);
        r.tail = (uint32_t)v[4] | ((unsigned long long)(uint32_t)v[5] << 32);
        r.status = (long long)(int32_t)(uint32_t)v[6];
        r.seq = seq;
    }

    ch->head = r.head;
    ch->tail = r.tail;
    if (r.status != HICR_OK) return (int)r.status;
    *n_out = r.k;
    if (push) {
        ctx->cnt[li].sent += r.k;
        ctx->cnt[ch->ring].recv += r.k;
    } else {
        ctx->cnt[ch->ring].sent += r.k;
        ctx->cnt[li].recv += r.k;
    }
    return HICR_OK;
}

int hicr_channel_push(hicr_channel_t *ch, hicr_slot_t src, uint64_t src_off, uint64_t n_tokens, uint64_t *n_pushed)
{
    return channel_call(ch, true, src, src_off, n_tokens, n_pushed);
}

int hicr_channel_pop(hicr_channel_t *ch, hicr_slot_t dst, uint64_t dst_off, uint64_t max_tokens, uint64_t *n_popped)
{
    return channel_call(ch, false, dst, dst_off, max_tokens, n_popped);
}

int hicr_channel_stream(hicr_channel_t *ch, hicr_slot_t src, uint64_t src_off, hicr_slot_t dst, uint64_t dst_off,
                        const uint64_t *batch_tokens, uint64_t n_batches)
{
    if (!ch || (!batch_tokens && n_batches)) return HICR_ERR_INVALID_ARG;
    hicr_ctx *ctx = ch->ctx;
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    const int64_t si = slot_find(ctx, src), di = slot_find(ctx, dst);
    if (si < 0 || di < 0) return HICR_ERR_INVALID_SLOT;
    if (ch->head != ch->tail) return HICR_ERR_INVALID_ARG;
    uint64_t total = 0;
    for (uint64_t i = 0; i < n_batches; i++) {
        if (batch_tokens[i] > (1ull << 48)) return HICR_ERR_OUT_OF_BOUNDS;
        total += batch_tokens[i];
        if (total > (1ull << 48)) return HICR_ERR_OUT_OF_BOUNDS;
    }
    const SlotRow &ss = ctx->rows[si], &ds = ctx->rows[di];
    if (!tokens_fit(total, ch->T, src_off, row_size(ss)) || !tokens_fit(total, ch->T, dst_off, row_size(ds)))
        return HICR_ERR_OUT_OF_BOUNDS;
    if (total == 0) return HICR_OK;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    int rc = channel_scratch(ch, n_batches * 8 + sizeof(PipeRing));
    if (rc != HICR_OK) return rc;
    uint64_t *d_batches = reinterpret_cast<uint64_t *>(ch->d_tab);
    HICR_CUDA(ctx, cudaMemcpyAsync(d_batches, batch_tokens, n_batches * 8, cudaMemcpyHostToDevice, ctx->stream));
    bool piped = false;
    {
        // 16 B-aligned shapes: the pipeline of bulk copies (hicr_pipe.cu), many pieces in flight per end
        PipeRing pr;
        pr.st = ch->d_state;
        pr.ring = reinterpret_cast<unsigned char *>(ctx->rows[ch->ring].base);
        pr.src = reinterpret_cast<const unsigned char *>(ss.base + src_off);
        pr.dst = reinterpret_cast<unsigned char *>(ds.base + dst_off);
        pr.count0 = ch->head;
        pr.id_ring = ch->ring;
        pr.id_src = (uint32_t)si;
        pr.id_dst = (uint32_t)di;
        pr.pad = 0;
        rc = pipe_run(ctx, &pr, reinterpret_cast<PipeRing *>(ch->d_tab + n_batches * 8), 1, ch->T, ch->C, total, d_batches, n_batches,
                      0, ctx->d_call, &piped);
        if (rc != HICR_OK) return rc;
    }
    if (!piped) {
        ChannelState *st = ch->d_state;
        unsigned char *ring = reinterpret_cast<unsigned char *>(ctx->rows[ch->ring].base);
        unsigned char *sp = reinterpret_cast<unsigned char *>(ss.base + src_off);
        unsigned char *dp = reinterpret_cast<unsigned char *>(ds.base + dst_off);
        uint64_t T = ch->T, C = ch->C;
        const uint64_t *bp = d_batches;
        unsigned long long *c0 = &ctx->d_cnt[si].sent, *c1 = &ctx->d_cnt[ch->ring].recv, *c2 = &ctx->d_cnt[ch->ring].sent,
                           *c3 = &ctx->d_cnt[di].recv;
        CallResult *res = ctx->d_call;
        void *args[] = {&st, &ring, &T, &C, &sp, &dp, &bp, &n_batches, &total, &c0, &c1, &c2, &c3, &res};
        HICR_CUDA(ctx, cudaLaunchCooperativeKernel((const void *)spsc_stream_kernel, dim3(2), dim3(kStreamThreads), args, 0,
                                                   ctx->stream));
        ctx->launches++;
        ctx->push_stale = true;
    }
    HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));   // also: batch_tokens has been consumed
    const CallResult r = read_result(ctx);
    ch->head = r.head;
    ch->tail = r.tail;
    ctx->cnt[si].sent += total;
    ctx->cnt[ch->ring].recv += total;
    ctx->cnt[ch->ring].sent += total;
    ctx->cnt[di].recv += total;
    return HICR_OK;
}

int hicr_mpsc_create(hicr_ctx_t *ctx, uint32_t producers, const hicr_slot_t *rings, uint64_t token_bytes,
                     uint64_t capacity, hicr_mpsc_t **out)
{
    if (!ctx || !out || !rings) return HICR_ERR_INVALID_ARG;
    *out = nullptr;
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    if (producers == 0 || token_bytes == 0 || capacity == 0) return HICR_ERR_INVALID_ARG;
    std::vector<uint32_t> idx(producers);
    for (uint32_t p = 0; p < producers; p++) {
        const int64_t ri = slot_find(ctx, rings[p]);
        if (ri < 0) return HICR_ERR_INVALID_SLOT;
        if (!tokens_fit(capacity, token_bytes, 0, row_size(ctx->rows[ri]))) return HICR_ERR_OUT_OF_BOUNDS;
        idx[p] = (uint32_t)ri;
    }
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    hicr_mpsc *m = new hicr_mpsc();
    m->ctx = ctx;
    m->P = producers;
    m->T = token_bytes;
    m->C = capacity;
    m->rings = idx;
    m->head.assign(producers, 0);
    m->tail.assign(producers, 0);
    cudaError_t e = cudaMalloc(&m->d_state, sizeof(ChannelState) * producers);
    if (e == cudaSuccess) e = cudaMemsetAsync(m->d_state, 0, sizeof(ChannelState) * producers, ctx->stream);
    if (e == cudaSuccess) e = cudaMalloc(&m->d_ptrs, (size_t)producers * (4 * 8 + 3 * 4));
    if (e == cudaSuccess) e = cudaMalloc(&m->d_pipe, (size_t)producers * sizeof(PipeRing));
    if (e != cudaSuccess) {
        cudaFree(m->d_state);
        cudaFree(m->d_ptrs);
        cudaFree(m->d_pipe);
        delete m;
        return cuda_fail(ctx, e, "hicr_mpsc_create");
    }
    for (uint32_t p = 0; p < producers; p++) ctx->ring_refs[idx[p]]++;
    *out = m;
    return HICR_OK;
}

int hicr_mpsc_destroy(hicr_mpsc_t *m)
{
    if (!m) return HICR_ERR_INVALID_ARG;
    if (m->ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    (void)cudaStreamSynchronize(m->ctx->stream);
    cudaFree(m->d_state);
    cudaFree(m->d_ptrs);
    cudaFree(m->d_pipe);
    for (auto r : m->rings) m->ctx->ring_refs[r]--;
    delete m;
    return HICR_OK;
}

int hicr_mpsc_counters(hicr_mpsc_t *m, uint32_t producer, uint64_t *head, uint64_t *tail)
{
    if (!m || !head || !tail || producer >= m->P) return HICR_ERR_INVALID_ARG;
    *head = m->head[producer];
    *tail = m->tail[producer];
    return HICR_OK;
}

int hicr_mpsc_stream(hicr_mpsc_t *m, const hicr_slot_t *src_slots, const uint64_t *src_offs, const hicr_slot_t *dst_slots,
                     const uint64_t *dst_offs, uint64_t tokens_per_producer, uint64_t max_batch)
{
    if (!m || !src_slots || !dst_slots || max_batch == 0) return HICR_ERR_INVALID_ARG;
    hicr_ctx *ctx = m->ctx;
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    const uint32_t P = m->P;
    const uint64_t N = tokens_per_producer;
    if (N > (1ull << 48) / m->T) return HICR_ERR_OUT_OF_BOUNDS;
    std::vector<uint64_t> ptrs(4 * (size_t)P);
    std::vector<uint32_t> ids(3 * (size_t)P);
    for (uint32_t p = 0; p < P; p++) {
        const int64_t si = slot_find(ctx, src_slots[p]), di = slot_find(ctx, dst_slots[p]);
        if (si < 0 || di < 0) return HICR_ERR_INVALID_SLOT;
        const uint64_t so = src_offs ? src_offs[p] : 0, dof = dst_offs ? dst_offs[p] : 0;
        if (!tokens_fit(N, m->T, so, row_size(ctx->rows[si])) || !tokens_fit(N, m->T, dof, row_size(ctx->rows[di])))
            return HICR_ERR_OUT_OF_BOUNDS;
        if (m->head[p] != m->tail[p]) return HICR_ERR_INVALID_ARG;
        ptrs[p] = ctx->rows[m->rings[p]].base;
        ptrs[P + p] = ctx->rows[si].base + so;
        ptrs[2 * P + p] = ctx->rows[di].base + dof;
        ptrs[3 * P + p] = m->tail[p];
        ids[p] = m->rings[p];
        ids[P + p] = (uint32_t)si;
        ids[2 * P + p] = (uint32_t)di;
    }
    if (N == 0) return HICR_OK;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    // 16 B-aligned shapes: the pipeline of bulk copies (hicr_pipe.cu), one producer CTA and one consumer
    // CTA per ring -- the single logical consumer is P CTAs
    bool piped = false;
    {
        std::vector<PipeRing> pr(P);
        for (uint32_t p = 0; p < P; p++) {
            pr[p].st = m->d_state + p;
            pr[p].ring = reinterpret_cast<unsigned char *>(ptrs[p]);
            pr[p].src = reinterpret_cast<const unsigned char *>(ptrs[P + p]);
            pr[p].dst = reinterpret_cast<unsigned char *>(ptrs[2 * P + p]);
            pr[p].count0 = m->tail[p];
            pr[p].id_ring = ids[p];
            pr[p].id_src = ids[P + p];
            pr[p].id_dst = ids[2 * P + p];
            pr[p].pad = 0;
        }
        int rc = pipe_run(ctx, pr.data(), m->d_pipe, P, m->T, m->C, N, nullptr, 0, max_batch, nullptr, &piped);
        if (rc != HICR_OK) return rc;
    }
    if (!piped) {
        // any other shape: vector copies, P producer CTAs and one consumer CTA whose warps share the rings;
        // co-residency of all P + 1 CTAs is what makes the spin-waits safe
        int per_sm = 0;
        HICR_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, mpsc_stream_kernel, kMpscThreads, 0));
        if ((uint64_t)per_sm * ctx->num_sms < (uint64_t)P + 1) return HICR_ERR_NO_CAPACITY;
        uint32_t *d_ids = reinterpret_cast<uint32_t *>(m->d_ptrs + 4 * (size_t)P);
        // (pageable sources: the runtime stages them before returning)
        HICR_CUDA(ctx, cudaMemcpyAsync(m->d_ptrs, ptrs.data(), ptrs.size() * 8, cudaMemcpyHostToDevice, ctx->stream));
        HICR_CUDA(ctx, cudaMemcpyAsync(d_ids, ids.data(), ids.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
        ChannelState *st = m->d_state;
        uint32_t Pv = P;
        uint64_t T = m->T, C = m->C, tok = N, mb = max_batch;
        const uint64_t *pp = m->d_ptrs;
        const uint32_t *ip = d_ids;
        SlotCnt *cnt = ctx->d_cnt;
        void *args[] = {&st, &Pv, &T, &C, &pp, &ip, &tok, &mb, &cnt};
        HICR_CUDA(ctx, cudaLaunchCooperativeKernel((const void *)mpsc_stream_kernel, dim3(P + 1), dim3(kMpscThreads), args, 0,
                                                   ctx->stream));
        ctx->launches++;
        ctx->push_stale = true;
    }
    HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (uint32_t p = 0; p < P; p++) {
        m->head[p] += N;
        m->tail[p] += N;
        ctx->cnt[ids[P + p]].sent += N;
        ctx->cnt[m->rings[p]].recv += N;
        ctx->cnt[m->rings[p]].sent += N;
        ctx->cnt[ids[2 * P + p]].recv += N;
    }
    return HICR_OK;
}

int hicr_mpsc_locking_stream(hicr_channel_t *ch, uint32_t producers, const hicr_slot_t *src_slots, hicr_slot_t dst,
                             uint64_t dst_off, uint64_t tokens_per_producer, uint64_t max_batch)
{
    if (!ch || !src_slots || producers == 0 || max_batch == 0) return HICR_ERR_INVALID_ARG;
    hicr_ctx *ctx = ch->ctx;
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    const uint32_t P = producers;
    const uint64_t N = tokens_per_producer;
    if (ch->head != ch->tail) return HICR_ERR_INVALID_ARG;   // requires an empty ring at entry
    const int64_t di = slot_find(ctx, dst);
    if (di < 0) return HICR_ERR_INVALID_SLOT;
    if (N > (1ull << 48) / ch->T / P) return HICR_ERR_OUT_OF_BOUNDS;
    std::vector<uint64_t> ptrs(P);
    std::vector<uint32_t> ids(P);
    for (uint32_t p = 0; p < P; p++) {
        const int64_t si = slot_find(ctx, src_slots[p]);
        if (si < 0) return HICR_ERR_INVALID_SLOT;
        if (!tokens_fit(N, ch->T, 0, row_size(ctx->rows[si]))) return HICR_ERR_OUT_OF_BOUNDS;
        ptrs[p] = ctx->rows[si].base;
        ids[p] = (uint32_t)si;
    }
    const SlotRow &ds = ctx->rows[di];
    if (!tokens_fit((uint64_t)P * N, ch->T, dst_off, row_size(ds))) return HICR_ERR_OUT_OF_BOUNDS;
    if (N == 0) return HICR_OK;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    // co-residency of all P + 1 CTAs is what makes the spin-waits (reservation, in-order commit) safe
    int per_sm = 0;
    HICR_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, mpsc_locking_kernel, kMpscThreads, 0));
    if ((uint64_t)per_sm * ctx->num_sms < (uint64_t)P + 1) return HICR_ERR_NO_CAPACITY;

    // scratch: [P] u64 source bases, one u64 reservation counter, [P] u32 table indices
    int rc = channel_scratch(ch, (size_t)P * 12 + 16);
    if (rc != HICR_OK) return rc;
    unsigned char *d_tab = ch->d_tab;
    uint64_t *d_ptrs = reinterpret_cast<uint64_t *>(d_tab);
    unsigned long long *d_reserve = reinterpret_cast<unsigned long long *>(d_tab + (size_t)P * 8);
    uint32_t *d_ids = reinterpret_cast<uint32_t *>(d_tab + (size_t)P * 8 + 8);
    const unsigned long long head0 = ch->head;
    HICR_CUDA(ctx, cudaMemcpyAsync(d_ptrs, ptrs.data(), (size_t)P * 8, cudaMemcpyHostToDevice, ctx->stream));
    HICR_CUDA(ctx, cudaMemcpyAsync(d_reserve, &head0, 8, cudaMemcpyHostToDevice, ctx->stream));
    HICR_CUDA(ctx, cudaMemcpyAsync(d_ids, ids.data(), (size_t)P * 4, cudaMemcpyHostToDevice, ctx->stream));
    {
        ChannelState *st = ch->d_state;
        uint32_t Pv = P, ring_slot = ch->ring, dst_slot = (uint32_t)di;
        unsigned char *ring = reinterpret_cast<unsigned char *>(ctx->rows[ch->ring].base);
        unsigned char *dp = reinterpret_cast<unsigned char *>(ds.base + dst_off);
        uint64_t T = ch->T, C = ch->C, tok = N, mb = max_batch;
        const uint64_t *pp = d_ptrs;
        const uint32_t *ip = d_ids;
        SlotCnt *cnt = ctx->d_cnt;
        CallResult *res = ctx->d_call;
        void *args[] = {&st, &d_reserve, &Pv, &ring, &T, &C, &pp, &ip, &dp, &tok, &mb, &cnt, &ring_slot, &dst_slot, &res};
        HICR_CUDA(ctx, cudaLaunchCooperativeKernel((const void *)mpsc_locking_kernel, dim3(P + 1), dim3(kMpscThreads), args, 0,
                                                   ctx->stream));
        ctx->launches++;
        ctx->push_stale = true;
    }
    HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const CallResult r = read_result(ctx);
    ch->head = r.head;
    ch->tail = r.tail;
    const uint64_t total = (uint64_t)P * N;
    for (uint32_t p = 0; p < P; p++) ctx->cnt[ids[p]].sent += N;
    ctx->cnt[ch->ring].recv += total;
    ctx->cnt[ch->ring].sent += total;
    ctx->cnt[di].recv += total;
    return HICR_OK;
}

}  // extern "C"
