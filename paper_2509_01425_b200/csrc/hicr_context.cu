// hicr_context.cu -- context, slot table (a1) and fence (a7) of the copy engine.
//
// a1  hicr_slot_register : "record the provided information and return a
//                          memory slot object"
// a7  hicr_fence         : "suspend execution until the expected number of
//                          incoming and outgoing data transfers have been completed"
#include "hicr_internal.cuh"

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

static int bad_to_status(unsigned id)
{
    switch (id) {
    case kBadInvalidSlot: return HICR_ERR_INVALID_SLOT;
    case kBadOutOfBounds: return HICR_ERR_OUT_OF_BOUNDS;
    case kBadNoCapacity: return HICR_ERR_NO_CAPACITY;
    default: return HICR_ERR_INVALID_ARG;
    }
}

// Read back the slot counters (device -> pinned -> host mirror) and wait for the stream.
int refresh_counters(hicr_ctx *ctx)
{
    const size_t n = ctx->slots.size();
    if (n == 0) return HICR_OK;
    unsigned char *p = ctx->h_fence;
    HICR_CUDA(ctx, cudaMemcpyAsync(p, ctx->d_sent, n * 8, cudaMemcpyDeviceToHost, ctx->stream));
    HICR_CUDA(ctx, cudaMemcpyAsync(p + 8 * (size_t)HICR_MAX_SLOTS, ctx->d_recv, n * 8, cudaMemcpyDeviceToHost,
                                   ctx->stream));
    HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    memcpy(ctx->sent.data(), p, n * 8);
    memcpy(ctx->recv.data(), p + 8 * (size_t)HICR_MAX_SLOTS, n * 8);
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
    const size_t n = ctx->slots.size();
    uint32_t words[kRwUsed];
    for (uint32_t k = 0; k < nb; k++) {
        const uint32_t b = k == 0 ? nb - 1 : k - 1;   // last batch first, then 0 .. nb-2
        const uint64_t seq = ctx->batch_seq - (nb - 1 - b);
        int rc = wait_words(ctx, ctx->h_rec[b].w, kRwUsed, rec_flag(seq), words);
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
        if (nb && n <= kPushSlots) {
            // the last batch pushed the cumulative counters next to the records
            int rc = wait_words(ctx, ctx->h_rec[kRecRing].w, n * kPushWordsPerSlot, rec_flag(ctx->batch_seq),
                                ctx->push_words.data());
            if (rc != HICR_OK) return rc;
            for (size_t s = 0; s < n; s++) {
                const uint32_t *w = ctx->push_words.data() + s * kPushWordsPerSlot;
                ctx->sent[s] = join64(w[0], w[1]);
                ctx->recv[s] = join64(w[2], w[3]);
            }
        } else {
            int rc = refresh_counters(ctx);
            if (rc != HICR_OK) return rc;
        }
    }
    for (auto &b : ctx->used_stage) ctx->free_stage.push_back(b);
    ctx->used_stage.clear();
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
    INIT_CUDA(cudaMemset(ctx->d_slots, 0xff, sizeof(SlotRow) * HICR_MAX_SLOTS));  // size = kInvalidSize
    INIT_CUDA(cudaMalloc(&ctx->d_sent, 8 * HICR_MAX_SLOTS));
    INIT_CUDA(cudaMalloc(&ctx->d_recv, 8 * HICR_MAX_SLOTS));
    INIT_CUDA(cudaMemset(ctx->d_sent, 0, 8 * HICR_MAX_SLOTS));
    INIT_CUDA(cudaMemset(ctx->d_recv, 0, 8 * HICR_MAX_SLOTS));
    INIT_CUDA(cudaMalloc(&ctx->d_ctl, sizeof(Ctl)));
    INIT_CUDA(cudaMemset(ctx->d_ctl, 0, sizeof(Ctl)));
    {
        // kRecRing records, then the pushed counter words (addressed as h_rec[kRecRing].w[...])
        const size_t rec_bytes = sizeof(HostRecord) * kRecRing + 8 * (size_t)kPushWordsPerSlot * kPushSlots;
        INIT_CUDA(cudaHostAlloc(&ctx->h_rec, rec_bytes, cudaHostAllocMapped));
        memset(ctx->h_rec, 0, rec_bytes);
        INIT_CUDA(cudaHostGetDevicePointer(&ctx->d_rec, ctx->h_rec, 0));
    }
    ctx->h_fence_bytes = 2 * 8 * (size_t)HICR_MAX_SLOTS;
    INIT_CUDA(cudaHostAlloc(&ctx->h_fence, ctx->h_fence_bytes, cudaHostAllocDefault));
    INIT_CUDA(cudaHostAlloc(&ctx->h_call, sizeof(CallResult) * 4, cudaHostAllocMapped));
    memset(ctx->h_call, 0, sizeof(CallResult) * 4);
    INIT_CUDA(cudaHostGetDevicePointer(&ctx->d_call, ctx->h_call, 0));
    for (int i = 0; i < 2; i++) INIT_CUDA(cudaEventCreate(&ctx->ev[i]));
    INIT_CUDA(cudaDeviceSynchronize());
#undef INIT_CUDA
    {
        int rc = engine_setup(ctx);
        if (rc != HICR_OK) {
            fprintf(stderr, "hicr_init: engine kernel cannot be made resident: %s\n", ctx->cuda_error.c_str());
            hicr_finalize(ctx);
            return rc;
        }
    }
    {
        // host threads for host-resident tables: the caller's plus helpers
        int threads = 4;
        const char *e = getenv("HICR_STAGE_THREADS");
        if (e && *e) threads = std::max(1, std::min(64, atoi(e)));
        ctx->stage_pool = stage_pool_create(threads - 1);
    }
    *out = ctx;
    return HICR_OK;
}

int hicr_finalize(hicr_ctx_t *ctx)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
    (void)cudaSetDevice(ctx->device);
    (void)cudaStreamSynchronize(ctx->stream);
#ifdef HICR_TRACE
    if (getenv("HICR_TRACE_FILE")) trace_dump(getenv("HICR_TRACE_FILE"));
#endif
    stage_pool_destroy(ctx->stage_pool);
    stage_done_free(ctx->stage_done);
    cudaFree(ctx->d_slots);
    cudaFree(ctx->d_sent);
    cudaFree(ctx->d_recv);
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
    if (size == kInvalidSize) return HICR_ERR_INVALID_ARG;
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
    if (ctx->slots.size() >= HICR_MAX_SLOTS) return HICR_ERR_NO_CAPACITY;
    SlotRow row{(uint64_t)(uintptr_t)dev_ptr, size};
    const size_t id = ctx->slots.size();
    // ordered after everything already enqueued on the stream; the row lives in pageable
    // host memory, so the runtime stages it before returning
    HICR_CUDA(ctx, cudaMemcpyAsync(ctx->d_slots + id, &row, sizeof(row), cudaMemcpyHostToDevice, ctx->stream));
    ctx->slots.push_back(row);
    ctx->sent.push_back(0);
    ctx->recv.push_back(0);
    ctx->ring_refs.push_back(0);
    ctx->registered_bytes += size;
    *out = (hicr_slot_t)id;
    return HICR_OK;
}

int hicr_slot_unregister(hicr_ctx_t *ctx, hicr_slot_t slot)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
    if (slot >= ctx->slots.size() || ctx->slots[slot].size == kInvalidSize) return HICR_ERR_INVALID_SLOT;
    if (ctx->ring_refs[slot]) return HICR_ERR_BUSY;
    SlotRow row{0, kInvalidSize};
    HICR_CUDA(ctx, cudaMemcpyAsync(ctx->d_slots + slot, &row, sizeof(row), cudaMemcpyHostToDevice, ctx->stream));
    ctx->registered_bytes -= ctx->slots[slot].size;
    ctx->slots[slot] = row;
    return HICR_OK;
}

int hicr_slot_counters(hicr_ctx_t *ctx, hicr_slot_t slot, uint64_t *sent, uint64_t *recv)
{
    if (!ctx || !sent || !recv) return HICR_ERR_INVALID_ARG;
    if (slot >= ctx->slots.size() || ctx->slots[slot].size == kInvalidSize) return HICR_ERR_INVALID_SLOT;
    *sent = ctx->sent[slot];
    *recv = ctx->recv[slot];
    return HICR_OK;
}

static int close_epoch(hicr_ctx *ctx);

int hicr_fence(hicr_ctx_t *ctx)
{
    if (!ctx) return HICR_ERR_INVALID_ARG;
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
    if (slot >= ctx->slots.size() || ctx->slots[slot].size == kInvalidSize) return HICR_ERR_INVALID_SLOT;
    auto reached = [&] { return ctx->sent[slot] >= sent && ctx->recv[slot] >= recv; };
    if (reached()) return HICR_OK;
    if (!ctx->epoch_open || ctx->batches_in_epoch == 0) return HICR_ERR_INVALID_ARG;   // nothing outstanding: never
    if (slot < kPushSlots && ctx->slots.size() <= kPushSlots) {
        // Every batch pushes the cumulative counters next to its completion record when its
        // copies are complete and visible: four flagged words per slot.  A snapshot whose four
        // flags agree comes from one batch; counters only grow, so the first such snapshot that
        // reaches the expected counts ends the wait.
        const unsigned long long *w = ctx->h_rec[kRecRing].w + (size_t)slot * kPushWordsPerSlot;
        const unsigned long long *last = ctx->h_rec[ctx->batches_in_epoch - 1].w;
        const uint32_t last_flag = rec_flag(ctx->batch_seq);
        unsigned spins = 0;
        for (;;) {
            uint32_t lf = 0;
            const bool last_done = word_ready(last + kRwUsed - 1, last_flag, &lf) && word_ready(last, last_flag, &lf);
            unsigned long long v[kPushWordsPerSlot];
            for (int k = 0; k < kPushWordsPerSlot; k++) v[k] = *reinterpret_cast<const volatile unsigned long long *>(w + k);
            const uint32_t f = (uint32_t)(v[0] >> 32);
            if (f != 0 && (uint32_t)(v[1] >> 32) == f && (uint32_t)(v[2] >> 32) == f && (uint32_t)(v[3] >> 32) == f) {
                const uint64_t sv = join64((uint32_t)v[0], (uint32_t)v[1]), rv = join64((uint32_t)v[2], (uint32_t)v[3]);
                if (sv >= ctx->sent[slot] && rv >= ctx->recv[slot]) {
                    ctx->sent[slot] = sv;
                    ctx->recv[slot] = rv;
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
