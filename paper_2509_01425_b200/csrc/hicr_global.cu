// hicr_global.cu -- Global Memory Slots: the local halves of the collective exchange, the
// mapping of other instances' storage, and the count exchange of the global fence
// (S3.1.4).
//
// "The exchange operation communicates the necessary metadata for remote instances to reach the
// associated memory slot": here a 256-byte handle with the slot's (tag, key),
// size, owner and the CUDA IPC handles of the allocation that holds it and of the owner's
// counter table.  Another context of the same process uses the owner's addresses as they are
// (peer access enabled if it sits on another device); another process maps them with
// cudaIpcOpenMemHandle.  Either way the global slot becomes one more row of this context's slot
// table (kind GLOBAL, hicr_internal.cuh), so hicr_memcpy_batch validates and copies it with the
// kernels it has: a put or a get is the initiator's copy over NVLink, nothing runs at the owner.
//
// The fence over instances follows SURVEY.md S8(e): local completion, then an exchange of what
// every instance initiated on every global slot, then the owner waits until its own device-side
// totals (which the initiators' kernels add to, data first) have reached the sums.
#include "hicr_internal.cuh"

#include <cuda.h>
#include <unistd.h>

#include <chrono>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <utility>

namespace hicr {

constexpr uint64_t kHandleMagic = 0x31304253524f4948ull;   // "HICRSB01"

// The bytes of hicr_global_handle_t.
struct HandleBody {
    uint64_t magic, tag, key, size;
    uint64_t owner_ctx;          // address of the owner's context in its process (identity, never dereferenced elsewhere)
    uint64_t base;               // the slot's address in the owner's process
    uint64_t base_offset;        // ... and its offset inside the allocation the IPC handle names
    uint64_t gcnt;               // address of the owner's counter entry for the slot, in the owner's process
    uint64_t gcnt_offset;
    uint32_t owner_instance, owner_slot, pid;
    int32_t device;
    uint32_t has_data_ipc, has_gcnt_ipc;
    cudaIpcMemHandle_t data_ipc, gcnt_ipc;
};
static_assert(sizeof(HandleBody) <= HICR_GLOBAL_HANDLE_BYTES, "the handle body fits the public struct");

struct GlobalSlot {
    uint64_t tag, key;
    uint32_t owner_instance;
    bool mine;                   // this context owns the storage
    uint32_t local_index;        // mine: table index of the local slot behind it
    std::string data_map, gcnt_map;   // keys of the IPC mappings it holds (empty: none)
};

struct GlobalTable {
    std::map<uint32_t, GlobalSlot> by_index;
    std::map<std::pair<uint64_t, uint64_t>, uint32_t> by_key;   // (tag, key) -> table index
    SlotCnt *h_gcnt = nullptr;   // pinned read-back of d_gcnt
};

// ---- IPC mappings of this process, shared by its contexts and counted
struct IpcMapping {
    void *base = nullptr;
    int device = 0;
    int refs = 0;
};
static std::mutex g_ipc_mu;
static std::map<std::string, IpcMapping> g_ipc;

static std::string ipc_key(uint32_t pid, const cudaIpcMemHandle_t &h, int device)
{
    std::string k(reinterpret_cast<const char *>(&pid), sizeof(pid));
    k.append(reinterpret_cast<const char *>(&device), sizeof(device));
    k.append(reinterpret_cast<const char *>(&h), sizeof(h));
    return k;
}

static int ipc_open(hicr_ctx *ctx, uint32_t pid, const cudaIpcMemHandle_t &h, std::string *key, void **base)
{
    std::lock_guard<std::mutex> lk(g_ipc_mu);
    *key = ipc_key(pid, h, ctx->device);
    IpcMapping &m = g_ipc[*key];
    if (m.refs == 0) {
        cudaError_t e = cudaIpcOpenMemHandle(&m.base, h, cudaIpcMemLazyEnablePeerAccess);
        if (e != cudaSuccess) {
            g_ipc.erase(*key);
            cuda_fail(ctx, e, "cudaIpcOpenMemHandle");
            return HICR_ERR_UNSUPPORTED_SPACE;   // the owner's memory space cannot be reached from this device
        }
        m.device = ctx->device;
    }
    m.refs++;
    *base = m.base;
    return HICR_OK;
}

static void ipc_close(const std::string &key)
{
    if (key.empty()) return;
    std::lock_guard<std::mutex> lk(g_ipc_mu);
    auto it = g_ipc.find(key);
    if (it == g_ipc.end()) return;
    if (--it->second.refs == 0) {
        int cur = 0;
        cudaGetDevice(&cur);
        cudaSetDevice(it->second.device);
        cudaIpcCloseMemHandle(it->second.base);
        cudaSetDevice(cur);
        (void)cudaGetLastError();
        g_ipc.erase(it);
    }
}

// Start of the allocation that holds `p` (what an IPC handle of `p` names).
static int allocation_base(hicr_ctx *ctx, uint64_t p, uint64_t *base)
{
    typedef CUresult (*range_fn)(CUdeviceptr *, size_t *, CUdeviceptr);
    static range_fn fn = nullptr;
    if (!fn) {
        void *f = nullptr;
        cudaDriverEntryPointQueryResult q;
        cudaError_t e = cudaGetDriverEntryPoint("cuMemGetAddressRange", &f, cudaEnableDefault, &q);
        if (e != cudaSuccess || !f) return cuda_fail(ctx, e == cudaSuccess ? cudaErrorUnknown : e, "cuMemGetAddressRange");
        fn = reinterpret_cast<range_fn>(f);
    }
    CUdeviceptr b = 0;
    size_t n = 0;
    if (fn(&b, &n, (CUdeviceptr)p) != CUDA_SUCCESS) {
        ctx->cuda_error = "cuMemGetAddressRange failed";
        return HICR_ERR_CUDA;
    }
    *base = (uint64_t)b;
    return HICR_OK;
}

int global_setup(hicr_ctx *ctx)
{
    ctx->globals = new GlobalTable();
    HICR_CUDA(ctx, cudaMalloc(&ctx->d_gcnt, sizeof(SlotCnt) * HICR_MAX_SLOTS));
    HICR_CUDA(ctx, cudaMemset(ctx->d_gcnt, 0, sizeof(SlotCnt) * HICR_MAX_SLOTS));
    HICR_CUDA(ctx, cudaMalloc(&ctx->d_gptr, sizeof(uint64_t) * HICR_MAX_SLOTS));
    HICR_CUDA(ctx, cudaMemset(ctx->d_gptr, 0, sizeof(uint64_t) * HICR_MAX_SLOTS));
    HICR_CUDA(ctx, cudaMalloc(&ctx->d_gdelta, sizeof(SlotCnt) * HICR_MAX_SLOTS));
    HICR_CUDA(ctx, cudaMemset(ctx->d_gdelta, 0, sizeof(SlotCnt) * HICR_MAX_SLOTS));
    HICR_CUDA(ctx, cudaHostAlloc(&ctx->globals->h_gcnt, sizeof(SlotCnt) * HICR_MAX_SLOTS, cudaHostAllocDefault));
    HICR_CUDA(ctx, cudaDeviceSynchronize());
    return HICR_OK;
}

void global_teardown(hicr_ctx *ctx)
{
    if (ctx->globals) {
        for (auto &kv : ctx->globals->by_index) {
            ipc_close(kv.second.data_map);
            ipc_close(kv.second.gcnt_map);
        }
        cudaFreeHost(ctx->globals->h_gcnt);
        delete ctx->globals;
        ctx->globals = nullptr;
    }
    cudaFree(ctx->d_gcnt);
    cudaFree(ctx->d_gptr);
    cudaFree(ctx->d_gdelta);
}

// hicr_slot_unregister of a row of kind GLOBAL: the kernels stop counting through it, its
// mappings are released, the local slot behind it (if this context owns it) is unpinned.
int global_forget(hicr_ctx *ctx, uint32_t index)
{
    GlobalTable *g = ctx->globals;
    auto it = g->by_index.find(index);
    if (it == g->by_index.end()) return HICR_OK;
    const uint64_t zero = 0;
    HICR_CUDA(ctx, cudaMemcpyAsync(ctx->d_gptr + index, &zero, sizeof(zero), cudaMemcpyHostToDevice, ctx->stream));
    HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));   // nothing in flight still reads the mapping
    ipc_close(it->second.data_map);
    ipc_close(it->second.gcnt_map);
    if (it->second.mine && ctx->ring_refs[it->second.local_index]) ctx->ring_refs[it->second.local_index]--;
    g->by_key.erase({it->second.tag, it->second.key});
    g->by_index.erase(it);
    ctx->n_global--;
    return HICR_OK;
}

}  // namespace hicr

using namespace hicr;

extern "C" {

int hicr_instance_set(hicr_ctx_t *ctx, uint32_t instance, uint32_t n_instances)
{
    if (!ctx || n_instances == 0 || instance >= n_instances) return HICR_ERR_INVALID_ARG;
    ctx->instance = instance;
    ctx->n_instances = n_instances;
    return HICR_OK;
}

int hicr_global_volunteer(hicr_ctx_t *ctx, uint64_t tag, uint64_t key, hicr_slot_t local_slot, hicr_global_handle_t *out)
{
    if (!ctx || !out) return HICR_ERR_INVALID_ARG;
    const int64_t i = slot_find(ctx, local_slot);
    if (i < 0) return HICR_ERR_INVALID_SLOT;
    const SlotRow &row = ctx->rows[i];
    if (row.meta & kRowGlobal) return HICR_ERR_INVALID_ARG;   // "volunteering zero or more local memory slots"
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    HandleBody h;
    memset(&h, 0, sizeof(h));
    h.magic = kHandleMagic;
    h.tag = tag;
    h.key = key;
    h.size = row_size(row);
    h.owner_ctx = (uint64_t)(uintptr_t)ctx;
    h.base = row.base;
    h.gcnt = (uint64_t)(uintptr_t)(ctx->d_gcnt + i);
    h.owner_instance = ctx->instance;
    h.owner_slot = local_slot;
    h.pid = (uint32_t)getpid();
    h.device = ctx->device;
    if (row.base && h.size) {
        uint64_t ab = 0;
        int rc = allocation_base(ctx, row.base, &ab);
        if (rc != HICR_OK) return rc;
        h.base_offset = row.base - ab;
        // (an allocation that cannot be shared -- e.g. from a virtual-memory pool -- still serves the
        // contexts of this process; another process then fails its exchange with UNSUPPORTED_SPACE)
        if (cudaIpcGetMemHandle(&h.data_ipc, reinterpret_cast<void *>(ab)) == cudaSuccess) h.has_data_ipc = 1;
        else (void)cudaGetLastError();
    }
    {
        uint64_t ab = 0;
        int rc = allocation_base(ctx, h.gcnt, &ab);
        if (rc != HICR_OK) return rc;
        h.gcnt_offset = h.gcnt - ab;
        if (cudaIpcGetMemHandle(&h.gcnt_ipc, reinterpret_cast<void *>(ab)) == cudaSuccess) h.has_gcnt_ipc = 1;
        else (void)cudaGetLastError();
    }
    memset(out->bytes, 0, sizeof(out->bytes));
    memcpy(out->bytes, &h, sizeof(h));
    return HICR_OK;
}

int hicr_global_exchange(hicr_ctx_t *ctx, uint64_t tag, const hicr_global_handle_t *handles, uint64_t n, hicr_slot_t *out_slots)
{
    if (!ctx || ((!handles || !out_slots) && n)) return HICR_ERR_INVALID_ARG;
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    if (n == 0) return HICR_OK;
    GlobalTable *g = ctx->globals;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    // ---- check everything first: the exchange creates all of its slots or none
    std::vector<HandleBody> hs(n);
    std::map<uint64_t, int> seen;
    for (uint64_t i = 0; i < n; i++) {
        memcpy(&hs[i], handles[i].bytes, sizeof(HandleBody));
        if (hs[i].magic != kHandleMagic || hs[i].tag != tag || hs[i].size > kSizeMask) return HICR_ERR_INVALID_ARG;
        if (seen[hs[i].key]++ || g->by_key.count({tag, hs[i].key})) return HICR_ERR_DUPLICATE_KEY;
    }
    const uint64_t free_rows = (uint64_t)ctx->free_idx.size() + (HICR_MAX_SLOTS - ctx->rows.size());
    if (n > free_rows) return HICR_ERR_NO_CAPACITY;
    const uint32_t pid = (uint32_t)getpid();
    uint64_t made = 0;
    int rc = HICR_OK;
    for (; made < n && rc == HICR_OK; made++) {
        const HandleBody &h = hs[made];
        GlobalSlot gs;
        gs.tag = tag;
        gs.key = h.key;
        gs.owner_instance = h.owner_instance;
        gs.mine = h.pid == pid && h.owner_ctx == (uint64_t)(uintptr_t)ctx;
        gs.local_index = h.owner_slot & kSlotIndexMask;
        uint64_t base = 0, gcnt = 0;
        if (h.pid == pid) {
            // the owner lives in this process: its addresses are ours ("Local Memory Slots ... within the
            // scope of a single HiCR instance" no longer)
            if (gs.mine && slot_find(ctx, h.owner_slot) < 0) rc = HICR_ERR_INVALID_SLOT;
            if (rc == HICR_OK && h.device != ctx->device) {
                cudaError_t e = cudaDeviceEnablePeerAccess(h.device, 0);
                if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) {
                    cuda_fail(ctx, e, "cudaDeviceEnablePeerAccess");
                    rc = HICR_ERR_UNSUPPORTED_SPACE;
                }
                (void)cudaGetLastError();
            }
            base = h.base;
            gcnt = h.gcnt;
        } else {
            void *m = nullptr;
            if (h.size && h.base) {
                if (!h.has_data_ipc) rc = HICR_ERR_UNSUPPORTED_SPACE;
                else rc = ipc_open(ctx, h.pid, h.data_ipc, &gs.data_map, &m);
                if (rc == HICR_OK) base = (uint64_t)(uintptr_t)m + h.base_offset;
            }
            if (rc == HICR_OK) {
                if (!h.has_gcnt_ipc) rc = HICR_ERR_UNSUPPORTED_SPACE;
                else rc = ipc_open(ctx, h.pid, h.gcnt_ipc, &gs.gcnt_map, &m);
                if (rc == HICR_OK) gcnt = (uint64_t)(uintptr_t)m + h.gcnt_offset;
            }
        }
        hicr_slot_t id = 0;
        if (rc == HICR_OK) rc = slot_install(ctx, base, h.size, kRowGlobal | (gs.mine ? 0 : kRowRemote), &id);
        if (rc == HICR_OK) {
            const uint32_t idx = id & kSlotIndexMask;
            cudaError_t e = cudaMemcpyAsync(ctx->d_gptr + idx, &gcnt, sizeof(gcnt), cudaMemcpyHostToDevice, ctx->stream);
            if (e != cudaSuccess) rc = cuda_fail(ctx, e, "cudaMemcpyAsync(gptr)");
            if (gs.mine) ctx->ring_refs[gs.local_index]++;   // the local slot stays registered while it is global
            g->by_index[idx] = gs;
            g->by_key[{tag, h.key}] = idx;
            ctx->n_global++;
            out_slots[made] = id;
        } else {
            ipc_close(gs.data_map);
            ipc_close(gs.gcnt_map);
            break;
        }
    }
    if (rc != HICR_OK) {
        for (uint64_t k = 0; k < made; k++) (void)hicr_slot_unregister(ctx, out_slots[k]);   // none, then
        return rc;
    }
    return HICR_OK;
}

int hicr_global_lookup(hicr_ctx_t *ctx, uint64_t tag, uint64_t key, hicr_slot_t *out)
{
    if (!ctx || !out) return HICR_ERR_INVALID_ARG;
    auto it = ctx->globals->by_key.find({tag, key});
    if (it == ctx->globals->by_key.end()) return HICR_ERR_INVALID_SLOT;
    *out = (hicr_slot_t)((ctx->gen[it->second] << kSlotIndexBits) | it->second);
    return HICR_OK;
}

int hicr_global_fence_begin(hicr_ctx_t *ctx, hicr_global_count_t *out, uint64_t cap, uint64_t *n)
{
    if (!ctx || !n || (!out && cap)) return HICR_ERR_INVALID_ARG;
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    GlobalTable *g = ctx->globals;
    *n = g->by_index.size();
    if (*n > cap) return HICR_ERR_NO_CAPACITY;   // before the fence: a retry with more room still gets the epoch's deferred error
    const int frc = hicr_fence(ctx);
    if (frc == HICR_ERR_CUDA) return frc;
    uint64_t k = 0;
    for (auto &kv : g->by_index) {
        out[k].tag = kv.second.tag;
        out[k].key = kv.second.key;
        out[k].sent = ctx->cnt[kv.first].sent;
        out[k].recv = ctx->cnt[kv.first].recv;
        k++;
    }
    return frc;
}

int hicr_global_fence_end(hicr_ctx_t *ctx, const hicr_global_count_t *all, uint64_t n_all, uint32_t timeout_ms)
{
    if (!ctx || (!all && n_all)) return HICR_ERR_INVALID_ARG;
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    GlobalTable *g = ctx->globals;
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    // the expected totals of every global slot this context owns: the sums of its lines
    std::map<uint32_t, SlotCnt> expect;   // local table index -> totals
    for (auto &kv : g->by_index)
        if (kv.second.mine) expect[kv.second.local_index] = SlotCnt{0, 0};
    for (uint64_t i = 0; i < n_all; i++) {
        auto it = g->by_key.find({all[i].tag, all[i].key});
        if (it == g->by_key.end()) continue;              // a slot this context does not know (another exchange)
        const GlobalSlot &gs = g->by_index[it->second];
        if (!gs.mine) continue;
        expect[gs.local_index].sent += all[i].sent;
        expect[gs.local_index].recv += all[i].recv;
    }
    if (expect.empty()) return HICR_OK;
    const size_t rows = ctx->rows.size();
    const auto t0 = std::chrono::steady_clock::now();
    for (;;) {
        HICR_CUDA(ctx, cudaMemcpyAsync(g->h_gcnt, ctx->d_gcnt, rows * sizeof(SlotCnt), cudaMemcpyDeviceToHost, ctx->stream));
        HICR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        bool ok = true;
        for (auto &kv : expect)
            ok = ok && g->h_gcnt[kv.first].sent >= kv.second.sent && g->h_gcnt[kv.first].recv >= kv.second.recv;
        if (ok) return HICR_OK;
        if (timeout_ms && std::chrono::steady_clock::now() - t0 > std::chrono::milliseconds(timeout_ms)) return HICR_ERR_TIMEOUT;
    }
}

int hicr_global_counters(hicr_ctx_t *ctx, hicr_slot_t slot, uint64_t *sent, uint64_t *recv)
{
    if (!ctx || !sent || !recv) return HICR_ERR_INVALID_ARG;
    if (ctx->capturing) return HICR_ERR_BUSY;   // a chain is being recorded on the stream (hicr_graph_begin)
    int64_t i = slot_find(ctx, slot);
    if (i < 0) return HICR_ERR_INVALID_SLOT;
    if (ctx->rows[i].meta & kRowGlobal) {
        auto it = ctx->globals->by_index.find((uint32_t)i);
        if (it == ctx->globals->by_index.end() || !it->second.mine) return HICR_ERR_INVALID_ARG;
        i = it->second.local_index;
    }
    HICR_CUDA(ctx, cudaSetDevice(ctx->device));
    SlotCnt c;
    HICR_CUDA(ctx, cudaMemcpy(&c, ctx->d_gcnt + i, sizeof(c), cudaMemcpyDeviceToHost));
    *sent = c.sent;
    *recv = c.recv;
    return HICR_OK;
}

}  // extern "C"
