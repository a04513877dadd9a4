// hicr_noalloc.cu -- hicr_memcpy_batch_noalloc: one batch of slot-to-slot copies for callers that
// cannot allocate device memory.
//
// Why it exists.  The context-based path (hicr_init / hicr_memcpy_batch) owns device memory: the
// slot table, the control block and, above all, the chunk queue that the engine kernel fills
// with the pieces of large descriptors -- and hicr_memcpy_batch frees and re-allocates that
// queue (cudaFree + cudaMalloc, both of which stall the whole device) the first time a batch is
// larger than any before it.  Some users of a copy engine cannot live with that:
//   - a process that handed all free HBM to a pool of its own at start-up (an inference server, a
//     framework's caching allocator): a later cudaMalloc from a library simply fails;
//   - a step loop with a latency budget and other streams in flight: cudaMalloc / cudaFree
//     synchronise the device, so a queue that grows in the middle of a run shows up as a
//     stall on streams that have nothing to do with the copy.
// For them this file carries the same operation -- validate every descriptor, expand the large
// ones into a queue of chunks, copy, count one message per descriptor on both slots
// -- as a variant of the engine whose queue, per-slot count histogram and
// control words live in ONE file-scope __device__ array of fixed size (g_scratch below, about
// 1 MiB; every GPU on which this library's code is loaded holds it until the process exits).
// The entry point calls no cudaMalloc, cudaFree, cudaHostAlloc or any library routine that
// allocates: one cudaMemsetAsync of the first 8.25 KiB of the array and two kernel launches on
// the caller's stream.
//
// What the caller has to know:
//   - Limits (hicr.h): HICR_NOALLOC_MAX_DESCS descriptors, HICR_NOALLOC_MAX_SLOTS slots; both are
//     checked on the host and refused with HICR_ERR_NO_CAPACITY.  The large descriptors of one call may
//     expand into at most HICR_NOALLOC_MAX_CHUNKS chunks of 128 KiB; that is only known on the
//     device and comes back in d_result like a validation error (nothing copied, nothing counted).
//   - First call on a device: the address of the array is looked up once per device
//     (cudaGetSymbolAddress, with that device current) and kept.  Make that first call before
//     any stream capture is under way.
//   - The array is shared by every call of the process on that device and keeps what the last
//     call left in it.  Each call clears, in stream order, the part that must start at zero.  Two
//     calls that overlap on the GPU (different streams, no dependency between them) race on it
//     and corrupt each other's queue: order them, e.g. by using one stream.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "hicr_internal.cuh"

namespace hicr {
namespace {

constexpr uint32_t kNaMaxDescs = HICR_NOALLOC_MAX_DESCS;
constexpr uint32_t kNaMaxSlots = HICR_NOALLOC_MAX_SLOTS;
constexpr uint32_t kNaMaxChunks = HICR_NOALLOC_MAX_CHUNKS;
constexpr int kNaMaxDevices = 64;

// Layout of the scratch array.  [0, kNaClearBytes) must be zero when the plan kernel starts.
struct NaCtl {
    unsigned long long bad_inv;   // atomicMax of ~((index << 4) | error id); 0 = every descriptor valid
    unsigned int n_chunk;         // items appended to the queue (may run past kNaMaxChunks: then bad_inv says so)
    unsigned int pad[61];
};
static_assert(sizeof(NaCtl) == 256, "control words take one 256-byte block");
constexpr size_t kNaHistOff = sizeof(NaCtl);                                      // [kNaMaxSlots][2] u32: sent, recv of this call
constexpr size_t kNaClearBytes = kNaHistOff + 2 * (size_t)kNaMaxSlots * sizeof(unsigned);
constexpr size_t kNaQueueOff = kNaClearBytes;                                     // kNaMaxChunks WorkItems
constexpr size_t kNaScratchBytes = kNaQueueOff + (size_t)kNaMaxChunks * sizeof(WorkItem);
static_assert(kNaQueueOff % 256 == 0, "queue starts on a 256-byte boundary");

// THE scratch memory.  In host code this name is only a handle for cudaGetSymbolAddress: it is not
// a device address and must never be handed to a kernel as one.
static __device__ __align__(256) unsigned char g_scratch[kNaScratchBytes];

struct NaArgs {
    const hicr_raw_slot_t *slots;
    uint32_t n_slots;
    const hicr_desc_t *descs;
    uint32_t n;
    unsigned char *scratch;       // device address of g_scratch, from cudaGetSymbolAddress
    unsigned long long *counters; // [n_slots][2] caller's cumulative sent / recv
    long long *result;            // [2] status, lowest bad index
};

__device__ __forceinline__ unsigned na_check_end(const hicr_raw_slot_t *slots, uint32_t n_slots, uint32_t id, uint64_t off,
                                                 uint64_t size, uint64_t *addr)
{
    if (id >= n_slots) return kBadInvalidSlot;
    const uint64_t sz = __ldg(&slots[id].size);
    if (off > sz || size > sz - off) return kBadOutOfBounds;
    *addr = (uint64_t)__ldg(reinterpret_cast<const unsigned long long *>(&slots[id].base)) + off;
    return 0;
}

// Kernel 1 of 2, one thread per descriptor: validate (destination before source, lowest bad
// index wins), count the batch's messages per slot into the scratch histogram (one atomic per
// distinct slot per warp), append the chunks of descriptors above kSmallMax to the scratch queue.
__global__ void __launch_bounds__(256) noalloc_plan_kernel(NaArgs a)
{
    NaCtl *ctl = reinterpret_cast<NaCtl *>(a.scratch);
    unsigned *hist = reinterpret_cast<unsigned *>(a.scratch + kNaHistOff);
    WorkItem *q = reinterpret_cast<WorkItem *>(a.scratch + kNaQueueOff);
    const unsigned lane = threadIdx.x & 31;
    for (uint32_t base = blockIdx.x * blockDim.x; base < a.n; base += gridDim.x * blockDim.x) {
        const uint32_t i = base + threadIdx.x;
        hicr_desc_t d = {};
        uint64_t dst = 0, src = 0;
        bool ok = false;
        if (i < a.n) {
            d = a.descs[i];
            unsigned bad = na_check_end(a.slots, a.n_slots, d.dst_slot, d.dst_off, d.size, &dst);
            if (!bad) bad = na_check_end(a.slots, a.n_slots, d.src_slot, d.src_off, d.size, &src);
            if (bad) atomicMax(&ctl->bad_inv, ~((unsigned long long)i << 4 | bad));
            ok = !bad;
        }
        const unsigned act = __ballot_sync(0xffffffffu, ok);
        if (!ok) continue;
        const unsigned md = __match_any_sync(act, d.dst_slot), ms = __match_any_sync(act, d.src_slot);
        if (lane == (unsigned)__ffs(ms) - 1) atomicAdd(&hist[2 * d.src_slot], (unsigned)__popc(ms));
        if (lane == (unsigned)__ffs(md) - 1) atomicAdd(&hist[2 * d.dst_slot + 1], (unsigned)__popc(md));
        if (d.size > kSmallMax) {
            const uint64_t nc64 = (d.size - 1) / kChunkBytes + 1;
            const unsigned nc = nc64 > kNaMaxChunks ? kNaMaxChunks + 1 : (unsigned)nc64;
            const unsigned at = atomicAdd(&ctl->n_chunk, nc);   // (at most 65,536 x 32,769: no wrap)
            if (at > kNaMaxChunks || nc > kNaMaxChunks - at) {
                atomicMax(&ctl->bad_inv, ~((unsigned long long)i << 4 | kBadNoCapacity));
            } else {
                for (unsigned c = 0; c < nc; c++) {
                    const uint64_t off = (uint64_t)c * kChunkBytes;
                    WorkItem w;
                    w.src = src + off;
                    w.dst = dst + off;
                    w.size = min(kChunkBytes, d.size - off);
                    w.pad = 0;
                    q[at + c] = w;
                }
            }
        }
    }
}

// Kernel 2 of 2.  A batch with any bad descriptor copies and counts nothing (reading 10) and only
// reports.  Otherwise: histogram added to the caller's counters, CTA per queued chunk, warp per
// small descriptor straight from the table.
__global__ void __launch_bounds__(256) noalloc_copy_kernel(NaArgs a)
{
    const NaCtl *ctl = reinterpret_cast<const NaCtl *>(a.scratch);
    const unsigned *hist = reinterpret_cast<const unsigned *>(a.scratch + kNaHistOff);
    const WorkItem *q = reinterpret_cast<const WorkItem *>(a.scratch + kNaQueueOff);
    const unsigned long long bad_inv = ctl->bad_inv;
    if (bad_inv) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            const unsigned long long bad = ~bad_inv;
            const unsigned id = (unsigned)(bad & 15);
            a.result[0] = id == kBadInvalidSlot ? HICR_ERR_INVALID_SLOT
                          : id == kBadOutOfBounds ? HICR_ERR_OUT_OF_BOUNDS
                                                  : HICR_ERR_NO_CAPACITY;
            a.result[1] = (long long)(bad >> 4);
        }
        return;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        a.result[0] = HICR_OK;
        a.result[1] = 0;
    }
    for (uint32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < 2 * a.n_slots; k += gridDim.x * blockDim.x) {
        const unsigned h = hist[k];
        if (h) a.counters[k] += h;
    }
    const unsigned n_chunk = ctl->n_chunk;
    for (unsigned c = blockIdx.x; c < n_chunk; c += gridDim.x) {
        const WorkItem w = q[c];
        copy_span<kUnroll, kLdStream, uint32_t, kUnrollShifted>(reinterpret_cast<unsigned char *>(w.dst),
                                                                reinterpret_cast<const unsigned char *>(w.src),
                                                                (uint32_t)w.size, (int)threadIdx.x, (int)blockDim.x);
    }
    const int lane = threadIdx.x & 31;
    const uint32_t warps = gridDim.x * (blockDim.x >> 5);
    for (uint32_t i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < a.n; i += warps) {
        const hicr_desc_t d = a.descs[i];
        if (d.size == 0 || d.size > kSmallMax) continue;
        const uint64_t dst = (uint64_t)__ldg(reinterpret_cast<const unsigned long long *>(&a.slots[d.dst_slot].base)) + d.dst_off;
        const uint64_t src = (uint64_t)__ldg(reinterpret_cast<const unsigned long long *>(&a.slots[d.src_slot].base)) + d.src_off;
        copy_span<kUnroll, kLdStream, uint32_t, kUnrollShifted>(reinterpret_cast<unsigned char *>(dst),
                                                                reinterpret_cast<const unsigned char *>(src),
                                                                (uint32_t)d.size, lane, 32);
    }
}

// Per device: the device address of g_scratch and the size of the copy kernel's grid, looked up by
// the first call on that device.
struct NaDevice {
    bool ready = false;
    unsigned char *scratch = nullptr;
    int copy_grid = 0;
};
NaDevice g_dev[kNaMaxDevices];
std::mutex g_dev_mutex;

// Called with `device` current.
int na_setup(int device, NaDevice **out)
{
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    NaDevice &nd = g_dev[device];
    if (!nd.ready) {
        unsigned char *p = nullptr;
        if (cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_scratch) != cudaSuccess || !p) return HICR_ERR_CUDA;
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || sms < 1) return HICR_ERR_CUDA;
        nd.scratch = p;
        nd.copy_grid = sms * 4;
        nd.ready = true;
    }
    *out = &nd;
    return HICR_OK;
}

int na_run(int device, cudaStream_t stream, NaArgs a)
{
    NaDevice *nd = nullptr;
    const int rc = na_setup(device, &nd);
    if (rc != HICR_OK) return rc;
    a.scratch = nd->scratch;
    if (cudaMemsetAsync(a.scratch, 0, kNaClearBytes, stream) != cudaSuccess) return HICR_ERR_CUDA;
    if (a.n) {
        const unsigned grid = (a.n + 255) / 256;
        noalloc_plan_kernel<<<grid, 256, 0, stream>>>(a);
        if (cudaGetLastError() != cudaSuccess) return HICR_ERR_CUDA;
    }
    noalloc_copy_kernel<<<nd->copy_grid, 256, 0, stream>>>(a);
    if (cudaGetLastError() != cudaSuccess) return HICR_ERR_CUDA;
    return HICR_OK;
}

}  // namespace
}  // namespace hicr

extern "C" int hicr_memcpy_batch_noalloc(int device, void *cuda_stream, const hicr_raw_slot_t *d_slots, uint32_t n_slots,
                                         const hicr_desc_t *d_descs, uint64_t n, uint64_t *d_counters, int64_t *d_result)
{
    using namespace hicr;
    if (device < 0 || device >= kNaMaxDevices || !d_result) return HICR_ERR_INVALID_ARG;
    if ((n_slots && (!d_slots || !d_counters)) || (n && !d_descs)) return HICR_ERR_INVALID_ARG;
    if (n > kNaMaxDescs || n_slots > kNaMaxSlots) return HICR_ERR_NO_CAPACITY;
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) return HICR_ERR_CUDA;
    if (prev != device && cudaSetDevice(device) != cudaSuccess) return HICR_ERR_CUDA;
    NaArgs a;
    a.slots = d_slots;
    a.n_slots = n_slots;
    a.descs = d_descs;
    a.n = (uint32_t)n;
    a.scratch = nullptr;
    a.counters = reinterpret_cast<unsigned long long *>(d_counters);
    a.result = reinterpret_cast<long long *>(d_result);
    const int rc = na_run(device, static_cast<cudaStream_t>(cuda_stream), a);
    if (prev != device) cudaSetDevice(prev);
    return rc;
}
