// hicr_context.cu -- context, slot table (a1) and fence (a7) of the copy engine.
//
// a1  hicr_slot_register : "record the provided information and return a
//                          memory slot object"
// a7  hicr_fence         : "suspend execution until the expected number of
//                          incoming and outgoing data transfers have been completed"
#include "hicr_internal.cuh"

#include <sched.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

namespace hicr {

int cuda_fail(hicr_ctx *ctx, cudaError_t e, const char *what)
{
    if (ctx) {
        ctx->cuda_error = std::string(cudaGetErrorName(e)) + ": " + cudaGetErrorString(e) + " in " + what;
    }
    (void)cudaGetLastError();  // clear the sticky-less error state
    return HICR_ERR_CUDA;
}

cudaError_t node_prepare(NodeLauncher &l, const void *func, dim3 grid, dim3 block, size_t smem, void **args, bool cooperative,
                         bool update)
{
    cudaKernelNodeParams p = {};
    p.func = const_cast<void *>(func);
    p.gridDim = grid;
    p.blockDim = block;
    p.sharedMemBytes = (unsigned)smem;
    p.kernelParams = args;
    cudaError_t e = cudaSuccess;
    if (!l.exec) {
        e = cudaGraphCreate(&l.graph, 0);
        if (e == cudaSuccess) e = cudaGraphAddKernelNode(&l.node, l.graph, nullptr, 0, &p);
        if (e == cudaSuccess && cooperative) {
            cudaKernelNodeAttrValue v;
            memset(&v, 0, sizeof(v));
            v.cooperative = 1;
            e = cudaGraphKernelNodeSetAttribute(l.node, cudaKernelNodeAttributeCooperative, &v);
        }
        if (e == cudaSuccess) e = cudaGraphInstantiate(&l.exec, l.graph, 0);
    } else if (update) {
        e = cudaGraphExecKernelNodeSetParams(l.exec, l.node, &p);
    }
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        node_free(l);
    }
    return e;
}

cudaError_t node_launch(NodeLauncher &l, const void *func, dim3 grid, dim3 block, size_t smem, void **args, bool cooperative,
                        bool update, cudaStream_t stream)
{
    cudaError_t e = node_prepare(l, func, grid, block, smem, args, cooperative, update);
    return e == cudaSuccess ? cudaGraphLaunch(l.exec, stream) : e;
}

void node_free(NodeLauncher &l)
{
    if (l.exec) cudaGraphExecDestroy(l.exec);
    if (l.graph) cudaGraphDestroy(l.graph);
    l = NodeLauncher();
}

int bad_to_status(unsigned id)
{
    switch (id) {
    case kBadInvalidSlot: return HICR_ERR_INVALID_SLOT;
    case kBadOutOfBounds: return HICR_ERR_OUT_OF_BOUNDS;
    case kBadNoCapacity: return HICR_ERR_NO_CAPACITY;
    case kBadDirection: return HICR_ERR_ILLEGAL_DIRECTION;
    default: return HICR_ERR_INVALID_ARG;
    }
}

// Read back the slot counters (device -> pinned -> host mirror) and wait for the stream: the
// fence's slow path, for everything the pushed snapshot of the last batch does not cover.
int refresh_counters(hicr_ctx *ctx)
{
    const size_t n = ctx->rows.size();
    if (n == 0) return HICR_OK;
    HICR_CUDA(ctx, cudaMemcpyAsync(ctx->h_fence, ctx->d_cnt, n * sizeof(SlotCnt), cudaMemcpyDeviceToHost, ctx->stream));
    HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    memcpy(ctx->cnt.data(), ctx->h_fence, n * sizeof(SlotCnt));
    return HICR_OK;
}

// One flagged word of a completion record (see HostRecord): true once it carries `flag`.
static inline bool word_ready(const unsigned long long *w, uint32_t flag, uint32_t *payload)
{
    const unsigned long long v = *reinterpret_cast<const volatile unsigned long long *>(w);
    if ((uint32_t)(v >> 32) != flag) return false;
    *payload = (uint32_t)v;
    return true;
}

// Wait until `n` flagged words starting at `w` all carry `flag`; payloads go to out[].
// Polls; every so often asks the stream, so that a faulted kernel turns into HICR_ERR_CUDA
// instead of a hang.
static int wait_words(hicr_ctx *ctx, const unsigned long long *w, size_t n, uint32_t flag, uint32_t *out)
{
    unsigned spins = 0;
    for (size_t i = 0; i < n; i++) {
        while (!word_ready(w + i, flag, out + i)) {
            if ((++spins & 0x3fff) == 0) {
                cudaError_t e = cudaStreamQuery(ctx->stream);
                if (e == cudaSuccess) {
                    if (word_ready(w + i, flag, out + i)) break;
                    ctx->cuda_error = "engine kernel finished without publishing its completion record";
                    return HICR_ERR_CUDA;
                }
                if (e != cudaErrorNotReady) return cuda_fail(ctx, e, "cudaStreamQuery(fence)");
            }
        }
    }
    return HICR_OK;
}

static inline uint64_t join64(uint32_t lo, uint32_t hi) { return (uint64_t)lo | ((uint64_t)hi << 32); }

// Complete everything enqueued so far in this epoch: wait for every batch's completion
// record (the last one first: stream order makes the earlier ones complete too), fold
// deferred errors into the epoch state, take the pushed counters and recycle staging.
// final_fence distinguishes hicr_fence from the internal drain that happens when an epoch
// issues more than kRecRing batches.
int drain_epoch(hicr_ctx *ctx, bool final_fence)
{
    const uint32_t nb = ctx->batches_in_epoch;
    const size_t n = ctx->rows.size();
    uint32_t words[kRwUsed];
    for (uint32_t k = 0; k < nb; k++) {
        const uint32_t b = k == 0 ? nb - 1 : k - 1;   // last batch first, then 0 .. nb-2
        const uint64_t seq = ctx->batch_seq - (nb - 1 - b);
        int rc = wait_words(ctx, ctx->h_rec[(seq - 1) % kRecRing].w, kRwUsed, rec_flag(seq), words);
        if (rc != HICR_OK) return rc;
        if (b == nb - 1) {
            ctx->last_t[0] = join64(words[kRwTStartLo], words[kRwTStartHi]);
            ctx->last_t[1] = join64(words[kRwTMidLo], words[kRwTMidHi]);
            ctx->last_t[2] = join64(words[kRwTEndLo], words[kRwTEndHi]);
        }
        ctx->rec_bad[b] = join64(words[kRwBadLo], words[kRwBadHi]);
    }
    for (uint32_t b = 0; b < nb; b++) {
        const unsigned long long bad_inv = ctx->rec_bad[b];
        if (bad_inv != 0 && ctx->epoch_error == HICR_OK) {
            const unsigned long long packed = ~bad_inv;
            ctx->epoch_error = bad_to_status((unsigned)(packed & 15));
            ctx->epoch_error_batch = ctx->epoch_batch_base + b;
            ctx->epoch_error_index = packed >> 4;
        }
    }
    ctx->epoch_batch_base += nb;
    ctx->batches_in_epoch = 0;
    if (n && final_fence) {
        // The last launched batch pushed the cumulative counters of the first last_n_push table
        // rows next to the records.  That snapshot serves the fence unless something counted, or
        // changed the table, after that launch (a channel kernel, a registration): then the
        // whole table is read back in stream order.
        if (ctx->batch_seq && !ctx->push_stale && n <= ctx->last_n_push) {
            int rc = wait_words(ctx, ctx->h_rec[kRecRing].w, n * kPushWordsPerSlot, rec_flag(ctx->batch_seq),
                                ctx->push_words.data());
            if (rc != HICR_OK) return rc;
            for (size_t s = 0; s < n; s++) {
                const uint32_t *w = ctx->push_words.data() + s * kPushWordsPerSlot;
                ctx->cnt[s].sent = join64(w[0], w[1]);
                ctx->cnt[s].recv = join64(w[2], w[3]);
            }
        } else {
            int rc = refresh_counters(ctx);
            if (rc != HICR_OK) return rc;
        }
    }
    // every batch of the epoch launched so far has completed, so has the staging it read
    for (auto &b : ctx->used_stage) ctx->free_stage.push_back(b);
    ctx->used_stage.clear();
    return HICR_OK;
}

// (a1) Put one row into the slot table: the lowest free index, under its next generation, with
// zeroed counters; stream-ordered after everything already enqueued.  flags = kRowGlobal / kRowRemote.
int slot_install(hicr_ctx *ctx, uint64_t base, uint64_t size, uint64_t flags, hicr_slot_t *out)
{
    if (ctx->capturing) return HICR_ERR_BUSY;
    uint32_t i;
    if (!ctx->free_idx.empty()) i = ctx->free_idx.back();
    else if (ctx->rows.size() < HICR_MAX_SLOTS) i = (uint32_t)ctx->rows.size();
    else return HICR_ERR_NO_CAPACITY;
    const bool reuse = i < ctx->rows.size();
    const uint32_t g = reuse ? ctx->gen[i] + 1 : 0;
    const SlotRow row{base, row_meta(size, g, flags)};
    // the row lives in pageable host memory, so the runtime stages it before returning
    HICR_CUDA(ctx, cudaMemcpyAsync(ctx->d_slots + i, &row, sizeof(row), cudaMemcpyHostToDevice, ctx->stream));
    if (reuse) {
        HICR_CUDA(ctx, cudaMemsetAsync(ctx->d_cnt + i, 0, sizeof(SlotCnt), ctx->stream));
        // owner-side totals of an earlier registration that was volunteered under this index: a new
        // slot starts at zero there too (an index never handed out before still is zero)
        if (ctx->d_gcnt) HICR_CUDA(ctx, cudaMemsetAsync(ctx->d_gcnt + i, 0, sizeof(SlotCnt), ctx->stream));
        ctx->free_idx.pop_back();
        ctx->rows[i] = row;
        ctx->gen[i] = g;
        ctx->cnt[i] = SlotCnt{0, 0};
        ctx->ring_refs[i] = 0;
        ctx->born[i] = ctx->batch_seq;
    } else {
        ctx->rows.push_back(row);
        ctx->gen.push_back(g);
        ctx->cnt.push_back(SlotCnt{0, 0});
        ctx->ring_refs.push_back(0);
        ctx->born.push_back(ctx->batch_seq);
    }
    ctx->registered_bytes += size;
    ctx->push_stale = true;
    ctx->table_version++;
    *out = (hicr_slot_t)((g << kSlotIndexBits) | i);
    return HICR_OK;
}

}  // namespace hicr

using namespace hicr;

extern "C" {

const char *hicr_strerror(int status)
{
    switch (status) {
    case HICR_OK: return "ok";
    case HICR_ERR_INVALID_ARG: return "invalid argument";
    case HICR_ERR_INVALID_SLOT: return "invalid memory slot";
    case HICR_ERR_OUT_OF_BOUNDS: return "range outside its memory slot";
    case HICR_ERR_UNSUPPORTED_SPACE: return "memory space not supported by this communication manager";
    case HICR_ERR_NO_CAPACITY: return "capacity exhausted";
    case HICR_ERR_CUDA: return "CUDA runtime error";
    case HICR_ERR_BUSY: return "object in use";
    case HICR_ERR_ILLEGAL_DIRECTION: return "global-to-global transfers are not permitted";
    default: return "unknown status";
    }
}

const char *hicr_last_cuda_error(hicr_ctx_t *ctx) { return ctx ? ctx->cuda_error.c_str() : ""; }

int hicr_init(hicr_ctx_t **out, int device, void *cuda_stream)
{
    if (!out) return HICR_ERR_INVALID_ARG;
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || count == 0) {
        (void)cudaGetLastError();
        return HICR_ERR_CUDA;  // no CPU fallback: the product path fails loudly without a GPU
    }
    if (device < 0 || device >= count) return HICR_ERR_INVALID_ARG;
    hicr_ctx *ctx = new hicr_ctx();
    ctx->device = device;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
#define INIT_CUDA(call)                                    \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) {                          \
            cuda_fail(ctx, e__, #call);                    \
            fprintf(stderr, "hicr_init: %s\n", ctx->cuda_error.c_str()); \
            hicr_finalize(ctx);                            \
            return HICR_ERR_CUDA;                          \
        }                                                  \
    } while (0)
    INIT_CUDA(cudaSetDevice(device));
    INIT_CUDA(cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, device));
    INIT_CUDA(cudaMalloc(&ctx->d_slots, sizeof(SlotRow) * HICR_MAX_SLOTS));
    INIT_CUDA(cudaMemset(ctx->d_slots, 0xff, sizeof(SlotRow) * HICR_MAX_SLOTS));  // meta = kInvalidMeta
    INIT_CUDA(cudaMalloc(&ctx->d_cnt, sizeof(SlotCnt) * HICR_MAX_SLOTS));
    INIT_CUDA(cudaMemset(ctx->d_cnt, 0, sizeof(SlotCnt) * HICR_MAX_SLOTS));
    INIT_CUDA(cudaMalloc(&ctx->d_ctl, sizeof(Ctl)));
    INIT_CUDA(cudaMemset(ctx->d_ctl, 0, sizeof(Ctl)));
    {
        // kRecRing records, then the pushed counter words (addressed as h_rec[kRecRing].w[...])
        const size_t rec_bytes = sizeof(HostRecord) * kRecRing + 8 * (size_t)kPushWordsPerSlot * kPushSlots;
        INIT_CUDA(cudaHostAlloc(&ctx->h_rec, rec_bytes, cudaHostAllocMapped));
        memset(ctx->h_rec, 0, rec_bytes);
        INIT_CUDA(cudaHostGetDevicePointer(&ctx->d_rec, ctx->h_rec, 0));
    }
    INIT_CUDA(cudaHostAlloc(&ctx->h_fence, sizeof(SlotCnt) * HICR_MAX_SLOTS, cudaHostAllocDefault));
    INIT_CUDA(cudaHostAlloc(&ctx->h_call, sizeof(CallResult) * 4, cudaHostAllocMapped));
    memset(ctx->h_call, 0, sizeof(CallResult) * 4);
    INIT_CUDA(cudaHostGetDevicePointer(&ctx->d_call, ctx->h_call, 0));
    for (int i = 0; i < 2; i++) INIT_CUDA(cudaEventCreate(&ctx->ev[i]));
    INIT_CUDA(cudaDeviceSynchronize());
#undef INIT_CUDA
    if (global_setup(ctx) != HICR_OK) {
        fprintf(stderr, "hicr_init: %s\n", ctx->cuda_error.c_str());
        hicr_finalize(ctx);
        return HICR_ERR_CUDA;
    }
    {
        int rc = engine_setup(ctx);
        if (rc != HICR_OK) {
            fprintf(stderr, "hicr_init: engine kernel cannot be made resident: %s\n", ctx->cuda_error.c_str());
            hicr_finalize(ctx);
            return rc;
        }
    }
    {
        // host threads for host-resident tables, beside the caller's: half the cores this process may run on
        cpu_set_t set;
        CPU_ZERO(&set);
        int cores = sched_getaffinity(0, sizeof(set), &set) == 0 ? CPU_COUNT(&set) : 1;
        ctx->stage_pool = stage_pool_create(std::max(1, std::min(kStageThreadsMax, cores / 2)) - 1);
    }
    *out = ctx;
    return HICR_OK;
}

int hicr_finalize(hicr_ctx_t *ctx)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
    (void)cudaSetDevice(ctx->device);
    (void)cudaStreamSynchronize(ctx->stream);
    stage_pool_destroy(ctx->stage_pool);
    stage_done_free(ctx->stage_done);
    global_teardown(ctx);
    launch_cache_free(ctx);
    cudaFree(ctx->d_slots);
    cudaFree(ctx->d_cnt);
    cudaFree(ctx->d_ctl);
    cudaFree(ctx->d_chunk);
    for (auto *v : {&ctx->free_stage, &ctx->used_stage})
        for (auto &b : *v) {
            cudaFreeHost(b.host);
            cudaFree(b.dev);
        }
    cudaFreeHost(ctx->h_fence);
    cudaFreeHost(ctx->h_rec);
    cudaFreeHost(ctx->h_call);
    for (int i = 0; i < 2; i++)
        if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    (void)cudaGetLastError();
    delete ctx;
    return HICR_OK;
}

int hicr_slot_register(hicr_ctx_t *ctx, void *dev_ptr, uint64_t size, hicr_slot_t *out)
{
    if (!ctx || !out) return HICR_ERR_INVALID_ARG;
    if (!dev_ptr && size) return HICR_ERR_INVALID_ARG;
    if (size > kSizeMask) return HICR_ERR_INVALID_ARG;
    if (dev_ptr) {
        // "If the communication manager supports communication between the memory spaces
        // ... Otherwise, it will be rejected": only this device's memory.
        cudaPointerAttributes a;
        cudaError_t e = cudaPointerGetAttributes(&a, dev_ptr);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            return HICR_ERR_UNSUPPORTED_SPACE;
        }
        if (a.type != cudaMemoryTypeDevice || a.device != ctx->device) return HICR_ERR_UNSUPPORTED_SPACE;
        if ((uint64_t)(uintptr_t)dev_ptr + size < (uint64_t)(uintptr_t)dev_ptr) return HICR_ERR_INVALID_ARG;
    }
    return slot_install(ctx, (uint64_t)(uintptr_t)dev_ptr, size, 0, out);
}

int hicr_slot_unregister(hicr_ctx_t *ctx, hicr_slot_t slot)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
    if (ctx->capturing) return HICR_ERR_BUSY;
    const int64_t i = slot_find(ctx, slot);
    if (i < 0) return HICR_ERR_INVALID_SLOT;
    if (ctx->ring_refs[i]) return HICR_ERR_BUSY;
    if (ctx->rows[i].meta & kRowGlobal) {
        int rc = global_forget(ctx, (uint32_t)i);   // unmap the owner's storage, unpin the local slot behind it
        if (rc != HICR_OK) return rc;
    }
    const SlotRow row{0, kInvalidMeta};
    HICR_CUDA(ctx, cudaMemcpyAsync(ctx->d_slots + i, &row, sizeof(row), cudaMemcpyHostToDevice, ctx->stream));
    ctx->registered_bytes -= row_size(ctx->rows[i]);
    ctx->rows[i] = row;
    ctx->push_stale = true;
    ctx->table_version++;
    // the index can be handed out again under the next generation (ids kept from before then name
    // nothing); an index that has used up its generations is retired
    if (ctx->gen[i] < kMaxGen) {
        auto &f = ctx->free_idx;
        f.insert(std::upper_bound(f.begin(), f.end(), (uint32_t)i, std::greater<uint32_t>()), (uint32_t)i);
    }
    return HICR_OK;
}

int hicr_slot_counters(hicr_ctx_t *ctx, hicr_slot_t slot, uint64_t *sent, uint64_t *recv)
{
    if (!ctx || !sent || !recv) return HICR_ERR_INVALID_ARG;
    const int64_t i = slot_find(ctx, slot);
    if (i < 0) return HICR_ERR_INVALID_SLOT;
    *sent = ctx->cnt[i].sent;
    *recv = ctx->cnt[i].recv;
    return HICR_OK;
}

static int close_epoch(hicr_ctx *ctx);

int hicr_fence(hicr_ctx_t *ctx)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
    if (ctx->capturing) return HICR_ERR_BUSY;
    if (!ctx->epoch_open) {
        // nothing outstanding: return at once
        ctx->last_error = HICR_OK;
        return HICR_OK;
    }
    int rc = drain_epoch(ctx, true);
    if (rc != HICR_OK) return rc;
    return close_epoch(ctx);
}

// Close the epoch as hicr_fence does once everything outstanding has been drained.
static int close_epoch(hicr_ctx *ctx)
{
    const int rc = ctx->epoch_error;
    ctx->last_error = rc;
    ctx->last_error_batch = ctx->epoch_error_batch;
    ctx->last_error_index = ctx->epoch_error_index;
    ctx->epoch_error = HICR_OK;
    ctx->epoch_batch_base = 0;
    ctx->epoch_open = false;
    return rc;
}

int hicr_fence_async(hicr_ctx_t *ctx)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
    // Batches are kernels on one stream: each starts after the one before it has completed, so
    // the ordering the fence promises holds already; only the bookkeeping of completion records,
    // deferred errors and counters is left open until the next blocking fence.
    return HICR_OK;
}

int hicr_fence_expected(hicr_ctx_t *ctx, hicr_slot_t slot, uint64_t sent, uint64_t recv)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
    if (ctx->capturing) return HICR_ERR_BUSY;
    const int64_t si = slot_find(ctx, slot);
    if (si < 0) return HICR_ERR_INVALID_SLOT;
    SlotCnt &c = ctx->cnt[si];
    auto reached = [&] { return c.sent >= sent && c.recv >= recv; };
    if (reached()) return HICR_OK;
    if (!ctx->epoch_open || ctx->batches_in_epoch == 0) return HICR_ERR_INVALID_ARG;   // nothing outstanding: never
    if (!ctx->push_stale && (uint64_t)si < ctx->last_n_push) {
        // Every batch pushes the cumulative counters next to its completion record when its
        // copies are complete and visible: four flagged words per slot.  A snapshot whose four
        // flags agree comes from one batch; counters only grow, so the first such snapshot that
        // reaches the expected counts ends the wait.
        const unsigned long long *w = ctx->h_rec[kRecRing].w + (size_t)si * kPushWordsPerSlot;
        const unsigned long long *last = ctx->h_rec[(ctx->batch_seq - 1) % kRecRing].w;
        const uint32_t last_flag = rec_flag(ctx->batch_seq);
        const uint64_t lo_seq = std::max(ctx->born[si], ctx->batch_seq - ctx->batches_in_epoch);
        unsigned spins = 0;
        for (;;) {
            uint32_t lf = 0;
            const bool last_done = word_ready(last + kRwUsed - 1, last_flag, &lf) && word_ready(last, last_flag, &lf);
            unsigned long long v[kPushWordsPerSlot];
            for (int k = 0; k < kPushWordsPerSlot; k++) v[k] = *reinterpret_cast<const volatile unsigned long long *>(w + k);
            const uint32_t f = (uint32_t)(v[0] >> 32);
            // ... and from a batch of this epoch launched after the slot took the index
            bool ours = false;
            for (uint64_t q = ctx->batch_seq; q > lo_seq && !ours; q--) ours = f == rec_flag(q);
            if (ours && (uint32_t)(v[1] >> 32) == f && (uint32_t)(v[2] >> 32) == f && (uint32_t)(v[3] >> 32) == f) {
                const uint64_t sv = join64((uint32_t)v[0], (uint32_t)v[1]), rv = join64((uint32_t)v[2], (uint32_t)v[3]);
                if (sv >= c.sent && rv >= c.recv) {
                    c.sent = sv;
                    c.recv = rv;
                }
                if (reached()) return HICR_OK;
            }
            if (last_done) break;   // everything enqueued has completed; look once more below
            if ((++spins & 0x3fff) == 0) {
                cudaError_t e = cudaStreamQuery(ctx->stream);
                if (e != cudaSuccess && e != cudaErrorNotReady) return cuda_fail(ctx, e, "cudaStreamQuery(fence_expected)");
            }
        }
    }
    // all outstanding work has completed (or the table is too large for pushed counters): an
    // ordinary fence, after which the counts either are there or never will be
    int rc = drain_epoch(ctx, true);
    if (rc != HICR_OK) return rc;
    rc = close_epoch(ctx);
    if (rc != HICR_OK) return rc;
    return reached() ? HICR_OK : HICR_ERR_INVALID_ARG;
}

int hicr_fence_error(hicr_ctx_t *ctx, uint64_t *batch_index, uint64_t *first_bad)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
    if (batch_index) *batch_index = ctx->last_error_batch;
    if (first_bad) *first_bad = ctx->last_error_index;
    return ctx->last_error;
}

int hicr_launch_count(hicr_ctx_t *ctx, uint64_t *launches)
{
    if (!ctx || !launches) return HICR_ERR_INVALID_ARG;
    *launches = ctx->launches;
    return HICR_OK;
}

int hicr_profile_enable(hicr_ctx_t *ctx, int on)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
    ctx->profiling = on != 0;
    ctx->ev_valid = false;
    return HICR_OK;
}

int hicr_profile_read(hicr_ctx_t *ctx, float *ms)
{
    if (!ctx || !ms) return HICR_ERR_INVALID_ARG;
    if (!ctx->ev_valid || ctx->epoch_open) return HICR_ERR_INVALID_ARG;   // only after a fence
    const uint64_t *t = ctx->last_t;
    ms[0] = (float)((double)(t[1] - t[0]) * 1e-6);
    ms[1] = (float)((double)(t[2] - t[1]) * 1e-6);
    ms[2] = (float)((double)(t[2] - t[0]) * 1e-6);
    HICR_CUDA(ctx, cudaEventSynchronize(ctx->ev[1]));
    HICR_CUDA(ctx, cudaEventElapsedTime(&ms[3], ctx->ev[0], ctx->ev[1]));
    return HICR_OK;
}

}  // extern "C"
