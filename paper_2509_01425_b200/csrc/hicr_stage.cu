// hicr_stage.cu -- host side of (a2) for host-resident descriptor tables: check every
// descriptor against the host mirror of the slot table while copying it into pinned
// staging, on a few host threads.
//
// One pass over a 2 MiB table is bound by host memory bandwidth (a plain memcpy of it takes
// as long as check + copy on one core of the GPU box), so the table is cut into pieces that
// the caller's thread and up to kStageThreadsMax - 1 helper threads claim from a shared cursor.  CUDA calls
// stay on the caller's thread: it sends every finished prefix of pieces to the device while
// the others are still being checked.  Helpers spin for a short while after a job (a loop of
// batches finds them awake) and then sleep on a condition variable.
#include "hicr_internal.cuh"

#include <atomic>
#include <chrono>
#include <condition_variable>
#include <mutex>
#include <thread>

namespace hicr {

struct StageJob {
    const hicr_desc_t *in = nullptr;
    hicr_desc_t *out = nullptr;
    uint64_t n = 0, piece = 0, n_pieces = 0;
    const SlotRow *rows = nullptr;
    size_t n_slots = 0;
    std::atomic<uint64_t> next{0};        // next piece to claim
    std::atomic<uint64_t> *done = nullptr;   // per piece: 0 = not yet, 1 = ok, 2 = has a bad descriptor
    std::atomic<uint64_t> large{0}, small{0}, small_bytes{0};
};

// One descriptor against the host mirror of the slot table, with THE validator the engine
// kernel uses for device-resident tables (check_transfer, hicr_internal.cuh).  0 or an error id.
static inline unsigned check_desc(const hicr_desc_t &d, const SlotRow *rows, size_t nslots)
{
    const uint32_t di = d.dst_slot & kSlotIndexMask, si = d.src_slot & kSlotIndexMask;
    const bool d_in = di < nslots, s_in = si < nslots;
    static const SlotRow none{0, kInvalidMeta};
    return check_transfer(d_in ? rows[di] : none, d_in, d.dst_slot, d.dst_off, s_in ? rows[si] : none, s_in, d.src_slot,
                          d.src_off, d.size);
}

// Claim one piece and do it; false if none is left.  A piece with a bad descriptor is marked
// and left (the caller rescans it for the lowest index); the others are complete in `out`.
static bool work_one(StageJob &j)
{
    const uint64_t p = j.next.fetch_add(1, std::memory_order_relaxed);
    if (p >= j.n_pieces) return false;
    const uint64_t i0 = p * j.piece, i1 = std::min(j.n, i0 + j.piece);
    uint64_t state = 1, nc = 0, ns = 0, sb = 0;
    for (uint64_t i = i0; i < i1; i++) {
        const hicr_desc_t d = j.in[i];
        if (check_desc(d, j.rows, j.n_slots) != 0) {
            state = 2;
            break;
        }
        if (d.size > kSmallMax) nc += d.size / kChunkBytes + 2;
        else if (d.size) {
            ns++;
            sb += d.size;
        }
        j.out[i] = d;
    }
    if (nc) j.large.fetch_add(nc, std::memory_order_relaxed);
    j.small.fetch_add(ns, std::memory_order_relaxed);
    j.small_bytes.fetch_add(sb, std::memory_order_relaxed);
    j.done[p].store(state, std::memory_order_release);
    return true;
}
static void work(StageJob &j)
{
    while (work_one(j)) {}
}

class StagePool {
public:
    explicit StagePool(int helpers)
    {
        for (int i = 0; i < helpers; i++) threads_.emplace_back([this] { loop(); });
    }
    ~StagePool()
    {
        {
            std::lock_guard<std::mutex> g(m_);
            stop_ = true;
        }
        cv_.notify_all();
        for (auto &t : threads_) t.join();
    }
    int helpers() const { return (int)threads_.size(); }
    // Publish a job to the helpers; the caller works on it too and calls finish() before
    // the job (and the caller's table) goes away.
    void start(StageJob *j)
    {
        job_.store(j, std::memory_order_release);
        epoch_.fetch_add(1, std::memory_order_acq_rel);
        if (sleepers_.load(std::memory_order_acquire) > 0) {
            std::lock_guard<std::mutex> g(m_);
            cv_.notify_all();
        }
    }
    // Store-buffering pattern with the helper's { active_++ ; job_.load }: both sides are
    // sequentially consistent, so either the helper sees nullptr or finish() sees it active.
    void finish()
    {
        job_.store(nullptr, std::memory_order_seq_cst);
        while (active_.load(std::memory_order_seq_cst) != 0) std::this_thread::yield();
    }

private:
    void loop()
    {
        uint64_t seen = 0;
        for (;;) {
            // spin for a while, then sleep
            const auto t0 = std::chrono::steady_clock::now();
            unsigned spins = 0;
            while (epoch_.load(std::memory_order_acquire) == seen) {
                if (stop_) return;
                if ((++spins & 1023) == 0 &&
                    std::chrono::steady_clock::now() - t0 > std::chrono::microseconds(kSpinUs)) {
                    std::unique_lock<std::mutex> g(m_);
                    sleepers_.fetch_add(1, std::memory_order_acq_rel);
                    cv_.wait(g, [&] { return stop_ || epoch_.load(std::memory_order_acquire) != seen; });
                    sleepers_.fetch_sub(1, std::memory_order_acq_rel);
                    if (stop_) return;
                }
            }
            seen = epoch_.load(std::memory_order_acquire);
            active_.fetch_add(1, std::memory_order_seq_cst);
            StageJob *j = job_.load(std::memory_order_seq_cst);
            if (j) work(*j);
            active_.fetch_sub(1, std::memory_order_acq_rel);
        }
    }
    static constexpr int kSpinUs = 1000;
    std::vector<std::thread> threads_;
    std::mutex m_;
    std::condition_variable cv_;
    std::atomic<uint64_t> epoch_{0};
    std::atomic<StageJob *> job_{nullptr};
    std::atomic<int> active_{0}, sleepers_{0};
    std::atomic<bool> stop_{false};
};

// Does the kernel read the staged table straight from pinned host memory (no copy to the device)?
// Short tables: yes (32 KiB over PCIe costs less than enqueueing a copy).  Long tables: only when they
// look like bulk pages -- 64 evenly spaced descriptors all between 2 KiB and kSmallMax bytes -- because
// then the copy phase is long enough to hide the descriptor fetches over PCIe behind it and the 2 MiB
// of config 2 need not cross the bus before the kernel may start (end to end 211 -> 185 us); small
// descriptors (config 4: 149 -> 154 us) and tables with large ones (3a: 3.53 -> 3.64 ms) keep the copy.
// A wrong guess costs time, never correctness: the kernel reads the same bytes either way.
bool table_read_in_place(const hicr_desc_t *descs, uint64_t n)
{
    if (n <= kZeroCopyDescs) return true;
    for (uint64_t k = 0; k < 64; k++) {
        const uint64_t sz = descs[k * (n / 64)].size;
        if (sz < 2048 || sz > kSmallMax) return false;
    }
    return true;
}

// (a2) for a host table: check + stage `descs` into the pinned block `b`, send it to b.dev on
// the context's stream.  Returns HICR_OK or a CUDA failure; *bad_status = HICR_OK or the status of
// the lowest bad index (*first_bad), with nothing to launch.  Totals: chunk-queue bound, small
// descriptors and their bytes.
int stage_table(hicr_ctx *ctx, const hicr_desc_t *descs, uint64_t n, const StageBlock &b, uint64_t *first_bad,
                int *bad_status, uint64_t *n_chunk_bound, uint64_t *n_small, uint64_t *small_bytes)
{
    constexpr uint64_t kPiece = 4096, kSendPieces = 4;
    const bool in_place = table_read_in_place(descs, n);
    StageJob j;
    j.in = descs;
    j.out = static_cast<hicr_desc_t *>(b.host);
    j.n = n;
    j.piece = kPiece;
    j.n_pieces = (n + kPiece - 1) / kPiece;
    j.rows = ctx->rows.data();
    j.n_slots = ctx->rows.size();
    if (ctx->stage_done_cap < j.n_pieces) {
        delete[] ctx->stage_done;
        ctx->stage_done = new std::atomic<uint64_t>[j.n_pieces];
        ctx->stage_done_cap = j.n_pieces;
    }
    j.done = ctx->stage_done;
    for (uint64_t p = 0; p < j.n_pieces; p++) j.done[p].store(0, std::memory_order_relaxed);
    const bool parallel = ctx->stage_pool && j.n_pieces >= 4;
    if (parallel) ctx->stage_pool->start(&j);

    int rc = HICR_OK;
    *bad_status = HICR_OK;
    uint64_t sent = 0, ready = 0;   // pieces sent to the device / checked prefix
    while (sent < j.n_pieces) {
        const bool worked = work_one(j);
        while (ready < j.n_pieces) {
            const uint64_t st = j.done[ready].load(std::memory_order_acquire);
            if (st == 0) break;
            if (st == 2) {
                // every earlier piece is clean, so the lowest bad index of the table is in here
                const uint64_t i0 = ready * kPiece, i1 = std::min(n, i0 + kPiece);
                for (uint64_t i = i0; i < i1 && *bad_status == HICR_OK; i++) {
                    const unsigned bad = check_desc(descs[i], j.rows, j.n_slots);
                    if (bad) {
                        *bad_status = bad_to_status(bad);
                        if (first_bad) *first_bad = i;
                    }
                }
                break;
            }
            ready++;
        }
        if (rc != HICR_OK || *bad_status != HICR_OK) break;
        if (in_place) {
            sent = ready;   // the kernel reads the pinned staging block in place (no copy to enqueue)
        } else if (ready - sent >= kSendPieces || (ready == j.n_pieces && ready > sent)) {
            const uint64_t i0 = sent * kPiece, i1 = std::min(n, ready * kPiece);
            cudaError_t e = cudaMemcpyAsync(static_cast<hicr_desc_t *>(b.dev) + i0, j.out + i0, (i1 - i0) * sizeof(hicr_desc_t),
                                            cudaMemcpyHostToDevice, ctx->stream);
            if (e != cudaSuccess) {
                rc = cuda_fail(ctx, e, "cudaMemcpyAsync(descriptor table)");
                break;
            }
            sent = ready;
        } else if (!worked) {
            std::this_thread::yield();   // the helpers hold the remaining pieces
        }
    }
    if (rc != HICR_OK || *bad_status != HICR_OK) j.next.store(j.n_pieces, std::memory_order_relaxed);   // nobody claims any more
    if (parallel) ctx->stage_pool->finish();
    *n_chunk_bound = j.large.load();
    *n_small = j.small.load();
    *small_bytes = j.small_bytes.load();
    return rc;
}

StagePool *stage_pool_create(int helpers) { return helpers > 0 ? new StagePool(helpers) : nullptr; }
void stage_pool_destroy(StagePool *p) { delete p; }
void stage_done_free(std::atomic<uint64_t> *p) { delete[] p; }

}  // namespace hicr
