// hicr_copy.cu -- hicr_memcpy_batch: descriptor ingest + validation (a2), binning and
// work expansion (a3), the two copy kernels (a4, a5) and counter accumulation (a6).
//
// The operation: the Communication Manager's memcpy, "specify the source and
// destination memory slots, as well as the offsets within them and the size of data to
// communicate ... the operation will be initiated. Otherwise, it will be rejected"
// (PAPER.md:373), batched; completion deferred to the fence.
//
// Per batch, on the context's stream:
//   plan_kernel        one thread per descriptor: validate against the slot table, resolve
//                      absolute addresses, classify by size, compact into the warp queue /
//                      expand into the chunk queue (warp ballot + warp prefix sums + one
//                      atomic per warp per queue), aggregate the per-slot message counts;
//                      the last CTA to finish commits the batch (go = 1, counts folded into
//                      the cumulative counters) iff no descriptor was invalid.
//   copy_small_kernel  persistent, one warp per queued descriptor of <= kSmallMax bytes.
//   copy_chunk_kernel  persistent, one CTA per kChunkBytes chunk of a larger descriptor.
// Both copy kernels do nothing unless go == 1, which makes the batch all-or-nothing.
#include "hicr_internal.cuh"

#include <algorithm>
#include <cstring>

namespace hicr {

__device__ __forceinline__ void report_bad(Ctl *ctl, uint64_t index, unsigned id)
{
    atomicMax(&ctl->bad_inv, ~((unsigned long long)index << 4 | id));
}

// (a2) + (a3) + (a6)
__global__ void __launch_bounds__(kPlanThreads)
plan_kernel(const hicr_desc_t *__restrict__ descs, uint64_t n, const SlotRow *__restrict__ slots, uint32_t n_slots,
            Ctl *ctl, WorkItem *__restrict__ small_q, uint64_t small_cap, WorkItem *__restrict__ chunk_q,
            uint64_t chunk_cap, unsigned int *pending, unsigned long long *sent, unsigned long long *recv)
{
    extern __shared__ unsigned int hist[];  // [2 * n_slots] when n_slots <= kSmemSlotHist
    const bool use_hist = n_slots <= kSmemSlotHist;
    if (use_hist) {
        for (uint32_t i = threadIdx.x; i < 2 * n_slots; i += blockDim.x) hist[i] = 0;
        __syncthreads();
    }
    const int lane = threadIdx.x & 31;
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = i < n;

    uint64_t src = 0, dst = 0, size = 0;
    uint32_t ss = 0, ds = 0;
    bool valid = false;
    if (active) {
        const uint4 *p = reinterpret_cast<const uint4 *>(descs + i);
        const uint4 lo = __ldg(p), hi = __ldg(p + 1);
        ds = lo.x;
        ss = lo.y;
        const uint64_t dst_off = (uint64_t)lo.z | ((uint64_t)lo.w << 32);
        const uint64_t src_off = (uint64_t)hi.x | ((uint64_t)hi.y << 32);
        size = (uint64_t)hi.z | ((uint64_t)hi.w << 32);
        // destination checked before source; overflow-safe "off + size <= slot size"
        unsigned bad = 0;
        SlotRow dr{0, kInvalidSize}, sr{0, kInvalidSize};
        if (ds < n_slots) dr = slots[ds];
        if (ss < n_slots) sr = slots[ss];
        if (dr.size == kInvalidSize) bad = kBadInvalidSlot;
        else if (dst_off > dr.size || size > dr.size - dst_off) bad = kBadOutOfBounds;
        else if (sr.size == kInvalidSize) bad = kBadInvalidSlot;
        else if (src_off > sr.size || size > sr.size - src_off) bad = kBadOutOfBounds;
        if (bad) report_bad(ctl, i, bad);
        else {
            valid = true;
            dst = dr.base + dst_off;
            src = sr.base + src_off;
        }
    }

    // ---- (a6) one message per descriptor: sent on the source slot, recv on the destination
    // (lanes with the same slot elect one leader; invalid lanes carry a key no slot has)
    {
        const unsigned ms = __match_any_sync(0xffffffffu, valid ? ss : 0xffffffffu);
        if (valid && lane == __ffs(ms) - 1) {
            if (use_hist) atomicAdd(&hist[ss], __popc(ms)); else atomicAdd(&pending[ss], __popc(ms));
        }
        const unsigned md = __match_any_sync(0xffffffffu, valid ? ds : 0xffffffffu);
        if (valid && lane == __ffs(md) - 1) {
            if (use_hist) atomicAdd(&hist[n_slots + ds], __popc(md));
            else atomicAdd(&pending[HICR_MAX_SLOTS + ds], __popc(md));
        }
    }

    // ---- (a3) binning: warp ballot + prefix sums, one atomic per warp per queue
    const bool is_small = valid && size <= kSmallMax;   // zero-size descriptors move nothing
    const bool is_large = valid && size > kSmallMax;
    const unsigned small_mask = __ballot_sync(0xffffffffu, is_small && size > 0);
    if (small_mask) {
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(&ctl->n_small, __popc(small_mask));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (is_small && size > 0) {
            const uint64_t pos = base + __popc(small_mask & ((1u << lane) - 1));
            if (pos < small_cap) {
                uint4 *q = reinterpret_cast<uint4 *>(small_q + pos);
                q[0] = make_uint4((unsigned)src, (unsigned)(src >> 32), (unsigned)dst, (unsigned)(dst >> 32));
                q[1] = make_uint4((unsigned)size, (unsigned)(size >> 32), 0, 0);
            } else report_bad(ctl, i, kBadNoCapacity);
        }
    }
    const unsigned large_mask = __ballot_sync(0xffffffffu, is_large);
    if (large_mask) {
        const unsigned nch = is_large ? (unsigned)((size + kChunkBytes - 1) / kChunkBytes) : 0u;
        // inclusive warp scan of the chunk counts
        unsigned incl = nch;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += v;
        }
        const unsigned total = __shfl_sync(0xffffffffu, incl, 31);
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(&ctl->n_chunk, total);
        base = __shfl_sync(0xffffffffu, base, 0);
        const uint64_t my_first = (uint64_t)base + (incl - nch);
        if (is_large && my_first + nch > chunk_cap) report_bad(ctl, i, kBadNoCapacity);
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
            if (first + cnt > chunk_cap) continue;
            for (unsigned c = lane; c < cnt; c += 32) {
                const uint64_t off = (uint64_t)c * kChunkBytes;
                const uint64_t len = min(kChunkBytes, sz - off);
                uint4 *q = reinterpret_cast<uint4 *>(chunk_q + first + c);
                const uint64_t s1 = s0 + off, d1 = d0 + off;
                q[0] = make_uint4((unsigned)s1, (unsigned)(s1 >> 32), (unsigned)d1, (unsigned)(d1 >> 32));
                q[1] = make_uint4((unsigned)len, (unsigned)(len >> 32), 0, 0);
            }
        }
    }

    // ---- flush the CTA histogram, then the last CTA commits or discards the batch
    if (use_hist) {
        __syncthreads();
        for (uint32_t s = threadIdx.x; s < 2 * n_slots; s += blockDim.x) {
            const unsigned v = hist[s];
            if (v) atomicAdd(&pending[s < n_slots ? s : HICR_MAX_SLOTS + (s - n_slots)], v);
        }
    }
    __threadfence();
    __syncthreads();
    __shared__ bool last;
    if (threadIdx.x == 0) last = atomicAdd(&ctl->done, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!last) return;
    __threadfence();
    const bool ok = *reinterpret_cast<volatile unsigned long long *>(&ctl->bad_inv) == 0;
    for (uint32_t s = threadIdx.x; s < n_slots; s += blockDim.x) {
        const unsigned a = __ldcg(&pending[s]), b = __ldcg(&pending[HICR_MAX_SLOTS + s]);
        if (a) {
            if (ok) sent[s] += a;
            pending[s] = 0;
        }
        if (b) {
            if (ok) recv[s] += b;
            pending[HICR_MAX_SLOTS + s] = 0;
        }
    }
    if (threadIdx.x == 0) ctl->go = ok ? 1u : 0u;
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

// (a4) one warp per descriptor of <= kSmallMax bytes
__global__ void __launch_bounds__(kCopyThreads)
copy_small_kernel(const Ctl *__restrict__ ctl, const WorkItem *__restrict__ q)
{
    if (__ldcg(&ctl->go) == 0) return;
    const unsigned n = __ldcg(&ctl->n_small);
    const int lane = threadIdx.x & 31;
    const unsigned warps = gridDim.x * (kCopyThreads / 32);
    unsigned i = blockIdx.x * (kCopyThreads / 32) + (threadIdx.x >> 5);
    if (i >= n) return;
    WorkItem w = load_item(q + i);
    while (true) {
        const unsigned nxt = i + warps;
        WorkItem wn;
        if (nxt < n) wn = load_item(q + nxt);   // fetch the next item while this one is copied
        copy_span<kUnroll, kLdStream>(reinterpret_cast<unsigned char *>(w.dst),
                                      reinterpret_cast<const unsigned char *>(w.src), w.size, lane, 32);
        if (nxt >= n) break;
        w = wn;
        i = nxt;
    }
}

// (a5) one CTA per chunk of a large descriptor
__global__ void __launch_bounds__(kCopyThreads)
copy_chunk_kernel(const Ctl *__restrict__ ctl, const WorkItem *__restrict__ q)
{
    if (__ldcg(&ctl->go) == 0) return;
    const unsigned n = __ldcg(&ctl->n_chunk);
    for (unsigned i = blockIdx.x; i < n; i += gridDim.x) {
        const WorkItem w = load_item(q + i);
        copy_span<kUnroll, kLdStream>(reinterpret_cast<unsigned char *>(w.dst),
                                      reinterpret_cast<const unsigned char *>(w.src), w.size, threadIdx.x,
                                      kCopyThreads);
    }
}

static int ensure_queues(hicr_ctx *ctx, uint64_t n)
{
    if (n > ctx->small_cap) {
        uint64_t cap = std::max<uint64_t>(n, 4096);
        cap = std::max(cap, ctx->small_cap * 2);
        HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (ctx->d_small) HICR_CUDA(ctx, cudaFree(ctx->d_small));
        ctx->d_small = nullptr;
        ctx->small_cap = 0;
        HICR_CUDA(ctx, cudaMalloc(&ctx->d_small, cap * sizeof(WorkItem)));
        ctx->small_cap = cap;
    }
    // With pairwise-disjoint destinations (the epoch precondition) a batch expands into
    // at most n + registered_bytes / kChunkBytes chunks.
    const uint64_t need = n + ctx->registered_bytes / kChunkBytes + 64;
    if (need > ctx->chunk_cap) {
        uint64_t cap = std::max(need, ctx->chunk_cap * 2);
        HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (ctx->d_chunk) HICR_CUDA(ctx, cudaFree(ctx->d_chunk));
        ctx->d_chunk = nullptr;
        ctx->chunk_cap = 0;
        HICR_CUDA(ctx, cudaMalloc(&ctx->d_chunk, cap * sizeof(WorkItem)));
        ctx->chunk_cap = cap;
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
    HICR_CUDA(ctx, cudaHostAlloc(&b.host, b.bytes, cudaHostAllocDefault));
    cudaError_t e = cudaMalloc(&b.dev, b.bytes);
    if (e != cudaSuccess) {
        cudaFreeHost(b.host);
        return cuda_fail(ctx, e, "cudaMalloc(stage)");
    }
    *out = b;
    return HICR_OK;
}

}  // namespace hicr

using namespace hicr;

extern "C" int hicr_memcpy_batch(hicr_ctx_t *ctx, const hicr_desc_t *descs, uint64_t n, int descs_on_device,
                                 uint64_t *first_bad)
{
    if (!ctx || (!descs && n)) return HICR_ERR_INVALID_ARG;
    if (n == 0) return HICR_OK;
    if (n >= (1ull << 32)) return HICR_ERR_NO_CAPACITY;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));

    uint64_t n_small_host = n, n_chunk_host = ~0ull;  // upper bounds used to size the grids
    const hicr_desc_t *d_descs = descs;
    if (!descs_on_device) {
        // (a2) host-resident table: validate here, all-or-nothing, lowest bad index
        uint64_t ns = 0, nc = 0;
        for (uint64_t i = 0; i < n; i++) {
            const hicr_desc_t &d = descs[i];
            int rc = HICR_OK;
            if (d.dst_slot >= ctx->slots.size() || ctx->slots[d.dst_slot].size == kInvalidSize)
                rc = HICR_ERR_INVALID_SLOT;
            else if (d.dst_off > ctx->slots[d.dst_slot].size || d.size > ctx->slots[d.dst_slot].size - d.dst_off)
                rc = HICR_ERR_OUT_OF_BOUNDS;
            else if (d.src_slot >= ctx->slots.size() || ctx->slots[d.src_slot].size == kInvalidSize)
                rc = HICR_ERR_INVALID_SLOT;
            else if (d.src_off > ctx->slots[d.src_slot].size || d.size > ctx->slots[d.src_slot].size - d.src_off)
                rc = HICR_ERR_OUT_OF_BOUNDS;
            if (rc != HICR_OK) {
                if (first_bad) *first_bad = i;
                return rc;
            }
            if (d.size > kSmallMax) nc += (d.size + kChunkBytes - 1) / kChunkBytes;
            else if (d.size) ns++;
        }
        n_small_host = ns;
        n_chunk_host = nc;
        StageBlock b;
        int rc = get_stage(ctx, n * sizeof(hicr_desc_t), &b);
        if (rc != HICR_OK) return rc;
        memcpy(b.host, descs, n * sizeof(hicr_desc_t));
        ctx->used_stage.push_back(b);
        HICR_CUDA(ctx, cudaMemcpyAsync(b.dev, b.host, n * sizeof(hicr_desc_t), cudaMemcpyHostToDevice, ctx->stream));
        d_descs = static_cast<const hicr_desc_t *>(b.dev);
    }

    if (ctx->batches_in_epoch == kCtlRing) {
        int rc = drain_epoch(ctx, false);
        if (rc != HICR_OK) return rc;
    }
    int rc = ensure_queues(ctx, n);
    if (rc != HICR_OK) return rc;
    if (n_chunk_host != ~0ull && n_chunk_host > ctx->chunk_cap) {
        // only possible when destinations overlap (precondition violated): refuse cleanly
        return HICR_ERR_NO_CAPACITY;
    }

    if (ctx->copy_ctas_per_sm == 0) {
        int a = 0, b = 0;
        HICR_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, copy_small_kernel, kCopyThreads, 0));
        HICR_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, copy_chunk_kernel, kCopyThreads, 0));
        ctx->copy_ctas_per_sm = std::max(1, std::min(a, b));
    }
    const uint32_t n_slots = (uint32_t)ctx->slots.size();
    Ctl *ctl = ctx->d_ctl + ctx->batches_in_epoch;
    const unsigned plan_grid = (unsigned)((n + kPlanThreads - 1) / kPlanThreads);
    const size_t hist_bytes = n_slots <= kSmemSlotHist ? 2 * (size_t)n_slots * sizeof(unsigned) : 0;
    const unsigned persistent = (unsigned)(ctx->num_sms * ctx->copy_ctas_per_sm);

    const bool prof = ctx->profiling;
    if (prof) HICR_CUDA(ctx, cudaEventRecord(ctx->ev[0], ctx->stream));
    plan_kernel<<<plan_grid, kPlanThreads, hist_bytes, ctx->stream>>>(
        d_descs, n, ctx->d_slots, n_slots, ctl, ctx->d_small, ctx->small_cap, ctx->d_chunk, ctx->chunk_cap,
        ctx->d_pending, ctx->d_sent, ctx->d_recv);
    ctx->launches++;
    if (prof) HICR_CUDA(ctx, cudaEventRecord(ctx->ev[1], ctx->stream));
    if (n_small_host) {
        const uint64_t want = (n_small_host + kCopyThreads / 32 - 1) / (kCopyThreads / 32);
        const unsigned grid = (unsigned)std::min<uint64_t>(want, persistent);
        copy_small_kernel<<<grid, kCopyThreads, 0, ctx->stream>>>(ctl, ctx->d_small);
        ctx->launches++;
    }
    if (prof) HICR_CUDA(ctx, cudaEventRecord(ctx->ev[2], ctx->stream));
    if (n_chunk_host) {
        const unsigned grid = (unsigned)std::min<uint64_t>(n_chunk_host, persistent);
        copy_chunk_kernel<<<grid, kCopyThreads, 0, ctx->stream>>>(ctl, ctx->d_chunk);
        ctx->launches++;
    }
    if (prof) {
        HICR_CUDA(ctx, cudaEventRecord(ctx->ev[3], ctx->stream));
        ctx->ev_valid = true;
    }
    HICR_CUDA(ctx, cudaGetLastError());
    ctx->batches_in_epoch++;
    ctx->epoch_open = true;
    return HICR_OK;
}
