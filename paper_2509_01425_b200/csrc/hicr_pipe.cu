// hicr_pipe.cu -- the device-resident channel runs as pipelines of bulk copies (a8, a9, a10).
//
// "Channels operate by exchanging pre-allocated circular buffers ... the producer knows where
// to push the next message, as long as the buffer has not filled up. At that point the producer
// may not send any more messages until the consumer notifies that a message has been consumed."
// (PAPER.md:642).  Non-locking MPSC: "dedicated buffers per producer".
//
// pipe_kernel moves `tokens` tokens through each of P rings: source -> ring -> sink.  A ring has
// two ENDS, each one CTA: CTA r < P is the producer of ring r, CTA P + r its consumer, so the
// single LOGICAL consumer of the MPSC set is P CTAs, one per ring; each ring's tail keeps a
// single writer side and each producer's order is kept (per-producer FIFO).  Head and tail are
// the 64-bit device counters of ChannelState; nothing else synchronises the two ends.
//
// Inside an end, the token stream is cut into PIECES -- at the ends of the pushes (the batch
// list of hicr_channel_stream, or every max_batch tokens), at every `piece_tokens` ring
// positions and where the ring wraps -- and piece g is moved by warp g mod W, whose lane 0
// drives 1-D bulk copies (TMA) through the warp's own two shared-memory stages:
//   producer  source -> stage (issued one piece ahead, it needs no room in the ring); when
//             tail shows room: stage -> ring, wait for the write to complete, then the head is
//             advanced by the piece with a release, pieces in order (a turn counter in shared
//             memory), so head = h always means "every token below h is in the ring";
//   consumer  when head covers the piece: ring -> stage; once it has landed the ring positions
//             are free: tail advanced with a release, pieces in order; then stage -> sink
//             without waiting (the sink is complete when the kernel ends).
// W warps keep W pieces of each end in flight, so an end is bound by bytes in flight over the
// ring round trip and not by one warp's copy latency.  The ring stays in L2; DRAM sees the
// source once and the sink once.
//
// Requires T % 16 == 0 and 16 B-aligned ring, source and sink addresses (bulk copies) and
// T <= the stage size; other shapes take the vector-copy kernels of hicr_channel.cu.
#include "hicr_internal.cuh"

#include <algorithm>
#include <cstdlib>

namespace hicr {

constexpr int kPipeStages = 2;            // shared-memory stages per warp
constexpr int kPipeMaxWarps = 28;

__device__ __forceinline__ void red_add_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long atom_add_u64(unsigned long long *p, unsigned long long v)
{
    unsigned long long old;
    asm volatile("atom.relaxed.gpu.global.add.u64 %0, [%1], %2;" : "=l"(old) : "l"(p), "l"(v) : "memory");
    return old;
}
__device__ __forceinline__ unsigned ld_acquire_cta_shared(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_cta_shared(unsigned *p, unsigned v)
{
    asm volatile("st.release.cta.shared::cta.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}

// The pieces of one end, in order.  t = tokens of the run before the piece, rp = its ring
// position, len = its tokens (never crossing a push end, a multiple of piece_tokens ring
// positions, or the wrap), g = its index.
struct PieceWalk {
    unsigned long long t, rp, rin, bend, bi;
    unsigned g, gmod;
};
struct Piece {
    unsigned long long t, rp;
    unsigned len, g;
};

struct PipeWalkCfg {
    unsigned long long tokens, C, max_batch;
    const unsigned long long *batches;   // producer of hicr_channel_stream: tokens per push; else nullptr
    unsigned pt, W;
    bool cut_pushes;                     // producer: pieces end where pushes end
};

__device__ __forceinline__ void walk_init(PieceWalk &w, const PipeWalkCfg &c, unsigned long long count0)
{
    w.t = 0;
    w.rp = count0 % c.C;
    w.rin = w.rp % c.pt;
    w.bi = 0;
    w.bend = !c.cut_pushes ? c.tokens : c.batches ? c.batches[0] : c.max_batch;
    w.g = 0;
    w.gmod = 0;
}

// Next piece of the end, or false when the run is through.
__device__ __forceinline__ bool walk_next(PieceWalk &w, const PipeWalkCfg &c, Piece &p)
{
    if (w.t >= c.tokens) return false;
    while (w.bend == w.t) {   // pushes of zero tokens, and the push that just ended
        w.bi++;
        w.bend += c.batches ? c.batches[w.bi] : c.max_batch;
    }
    const unsigned long long to_push_end = min(w.bend, c.tokens) - w.t;
    const unsigned long long to_ring_cut = min((unsigned long long)c.pt - w.rin, c.C - w.rp);
    const unsigned len = (unsigned)min(to_push_end, to_ring_cut);
    p.t = w.t;
    p.rp = w.rp;
    p.len = len;
    p.g = w.g;
    w.t += len;
    w.rp += len;
    w.rin += len;
    if (w.rp == c.C) w.rp = 0, w.rin = 0;
    if (w.rin == c.pt) w.rin = 0;
    w.g++;
    return true;
}

// Next piece that belongs to warp `warp` (pieces go round the warps).
__device__ __forceinline__ bool walk_next_own(PieceWalk &w, const PipeWalkCfg &c, unsigned warp, Piece &p)
{
    for (;;) {
        const unsigned owner = w.gmod;
        if (!walk_next(w, c, p)) return false;
        w.gmod = owner + 1 == c.W ? 0 : owner + 1;
        if (owner == warp) return true;
    }
}

struct PipeArgs {
    const PipeRing *rings;
    uint32_t P;
    uint32_t piece_tokens;
    uint32_t stage_bytes;
    unsigned long long T, C, tokens, max_batch;
    const unsigned long long *batches;
    SlotCnt *cnt;
    CallResult *res;                     // ring 0's head / tail at the end of the run (hicr_channel_stream)
};

__global__ void __launch_bounds__(kPipeMaxWarps * 32, 1) pipe_kernel(const PipeArgs a)
{
    extern __shared__ __align__(128) unsigned char dyn_smem[];   // [warp][stage][stage_bytes]
    __shared__ uint64_t bars[kPipeMaxWarps * kPipeStages];
    __shared__ unsigned turn;                                    // low 32 bits of the next piece to commit
    const int lane = threadIdx.x & 31;
    const unsigned warp = threadIdx.x >> 5, W = blockDim.x >> 5;
    const bool producer = blockIdx.x < a.P;
    const PipeRing r = a.rings[producer ? blockIdx.x : blockIdx.x - a.P];
    if (threadIdx.x == 0) turn = 0;
    if (lane == 0) {
        for (int s = 0; s < kPipeStages; s++) mbar_init(&bars[warp * kPipeStages + s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (lane != 0) return;   // one driver lane per warp: everything below is bulk-copy issue and waiting

    unsigned char *stage = dyn_smem + (size_t)warp * kPipeStages * a.stage_bytes;
    uint64_t *bar = &bars[warp * kPipeStages];
    PipeWalkCfg cfg;
    cfg.tokens = a.tokens;
    cfg.C = a.C;
    cfg.max_batch = a.max_batch;
    cfg.batches = a.batches;
    cfg.pt = a.piece_tokens;
    cfg.W = W;
    cfg.cut_pushes = producer;
    PieceWalk wk;
    walk_init(wk, cfg, r.count0);
    const unsigned long long T = a.T, C = a.C;
    ChannelState *st = r.st;
    unsigned k = 0;   // own pieces so far: stage k % 2, mbarrier parity (k / 2) & 1

    if (producer) {
        Piece cur, nxt;
        bool have = walk_next_own(wk, cfg, warp, cur);
        if (have) {
            mbar_expect_tx(bar, (unsigned)(cur.len * T));
            bulk_g2s(stage, r.src + cur.t * T, (unsigned)(cur.len * T), bar);
        }
        unsigned long long tail_seen = r.count0;   // tail only grows: a stale value is a safe bound
        while (have) {
            const unsigned s = k % kPipeStages, sn = (k + 1) % kPipeStages;
            const bool have_next = walk_next_own(wk, cfg, warp, nxt);
            if (have_next) {
                // the other stage is free: the store that last read it was waited for to completion
                mbar_expect_tx(bar + sn, (unsigned)(nxt.len * T));
                bulk_g2s(stage + (size_t)sn * a.stage_bytes, r.src + nxt.t * T, (unsigned)(nxt.len * T), bar + sn);
            }
            // room: every position of the piece has been popped ("as long as the buffer has not filled up")
            const unsigned long long end_abs = r.count0 + cur.t + cur.len;
            if (tail_seen + C < end_abs) {
                unsigned ns = 20;
                while ((tail_seen = ld_acquire(&st->tail)) + C < end_abs) {
                    __nanosleep(ns);
                    if (ns < 160) ns *= 2;
                }
            }
            fence_proxy_async();   // the acquire above (generic proxy) before the ring write (async proxy)
            mbar_wait(bar + s, (k / kPipeStages) & 1);
            bulk_s2g(r.ring + cur.rp * T, stage + (size_t)s * a.stage_bytes, (unsigned)(cur.len * T));
            bulk_commit();
            bulk_wait_all();       // the payload is written ...
            fence_proxy_async();   // ... ordered before what this thread does next ...
            __threadfence();       // ... and performed device-wide BEFORE the turn is taken: the fence is the slow
                                   // part of a release (0.8 us), and inside the turn it would serialise the pieces
            while (ld_acquire_cta_shared(&turn) != cur.g) {}
            red_add_u64(&st->head, cur.len);           // payload first, then the counter
            st_release_cta_shared(&turn, cur.g + 1);
            cur = nxt;
            have = have_next;
            k++;
        }
        return;
    }

    // ---- consumer end
    Piece cur;
    unsigned long long head_seen = r.count0;
    bool last = false;
    unsigned long long tail_end = 0;
    while (walk_next_own(wk, cfg, warp, cur)) {
        const unsigned s = k % kPipeStages;
        const unsigned long long end_abs = r.count0 + cur.t + cur.len;
        if (head_seen < end_abs) {
            unsigned ns = 20;
            while ((head_seen = ld_acquire(&st->head)) < end_abs) {
                __nanosleep(ns);
                if (ns < 160) ns *= 2;
            }
        }
        fence_proxy_async();                      // the acquire (generic proxy) before the ring read (async proxy)
        if (k >= kPipeStages) bulk_wait_read<kPipeStages - 1>();   // the sink store that last read this stage
        const unsigned bytes = (unsigned)(cur.len * T);
        mbar_expect_tx(bar + s, bytes);
        bulk_g2s(stage + (size_t)s * a.stage_bytes, r.ring + cur.rp * T, bytes, bar + s);
        mbar_wait(bar + s, (k / kPipeStages) & 1);
        // the ring positions have been read: "the consumer notifies that a message has been consumed"
        // (the wait on the mbarrier is an acquire: the reads are done before the counter moves)
        while (ld_acquire_cta_shared(&turn) != cur.g) {}
        const unsigned long long old = atom_add_u64(&st->tail, cur.len);
        st_release_cta_shared(&turn, cur.g + 1);
        bulk_s2g(r.dst + cur.t * T, stage + (size_t)s * a.stage_bytes, bytes);
        bulk_commit();
        if (cur.t + cur.len == a.tokens) {
            last = true;
            tail_end = old + cur.len;
        }
        k++;
    }
    bulk_wait_all();   // this warp's part of the sink is complete before the CTA may exit
    if (last) {
        // the ring is through: one message per token on every slot it touched (reading 15)
        atomicAdd(&a.cnt[r.id_src].sent, a.tokens);
        atomicAdd(&a.cnt[r.id_ring].recv, a.tokens);
        atomicAdd(&a.cnt[r.id_ring].sent, a.tokens);
        atomicAdd(&a.cnt[r.id_dst].recv, a.tokens);
        if (a.res && blockIdx.x == a.P) {
            a.res->k = a.tokens;
            a.res->head = ld_acquire(&st->head);
            a.res->tail = tail_end;
            a.res->status = HICR_OK;
            __threadfence_system();
        }
    }
}

// Shape of a run: warps per end, stage size, tokens per piece; false if the bulk-copy pipeline
// cannot take it (alignment, token larger than a stage, co-residency of 2 P CTAs).
struct PipeShape {
    unsigned warps, stage_bytes, piece_tokens;
    size_t smem;
};

static bool pipe_shape(hicr_ctx *ctx, uint32_t P, uint64_t T, PipeShape *out)
{
    if (T % 16 != 0 || T == 0) return false;
    int max_smem = 0;
    if (cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device) != cudaSuccess) return false;
    const unsigned per_sm = (2 * P + ctx->num_sms - 1) / ctx->num_sms;     // CTAs that must share an SM
    // shared memory of an SM, less 1 KiB per CTA the system keeps and the static part
    const size_t budget = std::min<size_t>((size_t)max_smem, (size_t)(228 * 1024) / per_sm - 2048);
    unsigned stage = 8192;
    while (stage > 1024 && (T > stage || budget < (size_t)2 * kPipeStages * stage)) stage /= 2;
    if (T > stage || budget < (size_t)kPipeStages * stage) return false;
    unsigned warps = (unsigned)std::min<size_t>(budget / ((size_t)kPipeStages * stage), P == 1 ? 12 : 6);
    // (experiments only; removed once the defaults are set from the sweep)
    if (const char *e = getenv("HICR_PIPE_W")) warps = (unsigned)std::max(1, atoi(e));
    if (const char *e = getenv("HICR_PIPE_STAGE")) stage = (unsigned)std::max(1024, atoi(e));
    warps = std::min<unsigned>(warps, kPipeMaxWarps);
    if (T > stage || warps < 1 || 32 * warps > 1024) return false;
    out->warps = warps;
    out->stage_bytes = stage;
    out->piece_tokens = (unsigned)(stage / T);
    out->smem = (size_t)warps * kPipeStages * stage;
    if (out->smem > (size_t)max_smem) return false;
    if (cudaFuncSetAttribute(pipe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)out->smem) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    int resident = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, pipe_kernel, (int)(32 * warps), out->smem) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return (uint64_t)resident * ctx->num_sms >= 2ull * P;   // both ends of every ring spin on each other
}

// Runs the pipeline if the shape allows it (*ran = true) on the context's stream; the caller
// synchronises.  h_rings: P host records; d_rings: device space for them; d_batches: the push
// sizes on the device, or nullptr for pushes of max_batch tokens.
int pipe_run(hicr_ctx *ctx, const PipeRing *h_rings, PipeRing *d_rings, uint32_t P, uint64_t T, uint64_t C, uint64_t tokens,
             const uint64_t *d_batches, uint64_t max_batch, CallResult *res, bool *ran)
{
    *ran = false;
    PipeShape sh;
    for (uint32_t p = 0; p < P; p++) {
        const uintptr_t bits = (uintptr_t)h_rings[p].ring | (uintptr_t)h_rings[p].src | (uintptr_t)h_rings[p].dst;
        if (bits % 16) return HICR_OK;
    }
    if (!pipe_shape(ctx, P, T, &sh)) return HICR_OK;
    HICR_CUDA(ctx, cudaMemcpyAsync(d_rings, h_rings, sizeof(PipeRing) * P, cudaMemcpyHostToDevice, ctx->stream));
    PipeArgs a;
    a.rings = d_rings;
    a.P = P;
    a.piece_tokens = sh.piece_tokens;
    a.stage_bytes = sh.stage_bytes;
    a.T = T;
    a.C = C;
    a.tokens = tokens;
    a.max_batch = max_batch;
    a.batches = reinterpret_cast<const unsigned long long *>(d_batches);
    a.cnt = ctx->d_cnt;
    a.res = res;
    void *args[] = {&a};
    HICR_CUDA(ctx, cudaLaunchCooperativeKernel((const void *)pipe_kernel, dim3(2 * P), dim3(32 * sh.warps), args, sh.smem,
                                               ctx->stream));
    ctx->launches++;
    ctx->push_stale = true;
    *ran = true;
    return HICR_OK;
}

}  // namespace hicr
