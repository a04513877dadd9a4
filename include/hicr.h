/*
 * hicr.h -- C ABI of the B200-native HiCR memory-slot copy engine and token channels.
 *
 * What this library is: the data-parallel hot path of the HiCR runtime-support-layer
 * model (arxiv 2509.01425, cited below as PAPER.md:<line>), i.e. the Communication
 * Manager's `memcpy` between registered Local Memory Slots, completed by `fence`
 * (listing PAPER.md:524-535), plus the Channels frontend's
 * fixed-size-token circular buffer, plus Global Memory Slots: slots
 * exchanged between instances and reached by put / get.  One context =
 * one GPU's HBM as its memory space; other instances' slots are reached over CUDA IPC peer
 * mappings.  Every step of the path runs in hand-written sm_100a CUDA kernels;
 * there is no CPU fallback: without a CUDA device every call returns HICR_ERR_CUDA.
 *
 * Conventions
 *   - C linkage, `int` status return (HICR_OK = 0, errors negative), no exceptions and
 *     no callbacks cross the boundary.
 *   - All sizes and offsets are bytes, uint64_t (SURVEY.md S8(c) reading 2).
 *   - "device pointer" = an address in the memory of the device given to hicr_init;
 *     "host pointer" = ordinary host memory.  Each argument says which it is.
 *   - The library never owns slot storage (it "will record the provided
 *     information"); the caller keeps it alive until hicr_slot_unregister/hicr_finalize.
 *   - All device work is enqueued on the cudaStream_t given to hicr_init.
 *   - A context and its channels are driven by one host thread at a time.
 */
#ifndef HICR_H
#define HICR_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes -------------------------------------------------------------- */
#define HICR_OK                     0
#define HICR_ERR_INVALID_ARG      (-1)  /* NULL where a pointer is required, capacity 0, ... */
#define HICR_ERR_INVALID_SLOT     (-2)  /* slot id not registered (or unregistered twice)    */
#define HICR_ERR_OUT_OF_BOUNDS    (-3)  /* off > slot size or size > slot size - off         */
#define HICR_ERR_UNSUPPORTED_SPACE (-4) /* pointer is not memory of this device: "Otherwise,
                                           it will be rejected"               */
#define HICR_ERR_NO_CAPACITY      (-5)  /* slot table / work queue / allocation exhausted    */
#define HICR_ERR_CUDA             (-6)  /* a CUDA runtime call failed; hicr_last_cuda_error  */
#define HICR_ERR_BUSY             (-7)  /* object still referenced (e.g. slot used by a channel) */
#define HICR_ERR_ILLEGAL_DIRECTION (-8) /* "Global-to-Global operations are not permitted"
                                                                               */
#define HICR_ERR_DUPLICATE_KEY    (-9)  /* a (tag, key) pair names one global slot */
#define HICR_ERR_TIMEOUT         (-10)  /* a global fence did not see the expected counts in time */

typedef struct hicr_ctx hicr_ctx_t;          /* opaque context  */
typedef struct hicr_channel hicr_channel_t;  /* opaque SPSC channel */
typedef struct hicr_mpsc hicr_mpsc_t;        /* opaque non-locking MPSC channel set */
typedef uint32_t hicr_slot_t;                /* slot id, valid for one context: dense (0, 1, 2, ...) until
                                                ids are recycled -- {generation:20 | table index:12},
                                                an unregistered id is never valid again */

#define HICR_MAX_SLOTS 4096u

/* One transfer.  Field order follows the paper's call
 *   cmm->memcpy(dst, 0, message, 0, messageSize)
 * i.e. destination slot, destination offset, source slot, source offset, size.
 * 32 bytes, little endian, no padding. */
typedef struct hicr_desc {
    uint32_t dst_slot;
    uint32_t src_slot;
    uint64_t dst_off;
    uint64_t src_off;
    uint64_t size;
} hicr_desc_t;

/* ---- context (plumbing) ----------------------------------------------------------- */

/* Create a context on CUDA device `device`; all work goes to `cuda_stream` (a
 * cudaStream_t passed as void*; NULL = the legacy default stream).  *out receives the
 * context.  The context owns the device-side slot table, work queues, control blocks
 * and staging buffers.  Errors: HICR_ERR_INVALID_ARG, HICR_ERR_CUDA (no device). */
int hicr_init(hicr_ctx_t **out, int device, void *cuda_stream);

/* Wait for outstanding work, free everything the context owns (never slot storage). */
int hicr_finalize(hicr_ctx_t *ctx);

/* Static text for a status code. */
const char *hicr_strerror(int status);

/* Text of the last CUDA runtime error seen by this context ("" if none). Host pointer,
 * owned by the context. */
const char *hicr_last_cuda_error(hicr_ctx_t *ctx);

/* ---- memory slots ------------------------------------------- */

/* Register an existing device allocation [dev_ptr, dev_ptr + size) as a Local Memory
 * Slot: "manual registration of an existing memory allocation as a new local memory
 * slot by specifying its address, size".  Any base alignment; size 0 is
 * allowed (then dev_ptr may be NULL).  Sent/received counters start at 0.  *out
 * receives a dense id.  Errors: HICR_ERR_UNSUPPORTED_SPACE if dev_ptr is not device
 * memory of this context's device; HICR_ERR_NO_CAPACITY beyond HICR_MAX_SLOTS live
 * slots (an unregistered slot's table index is handed out again, under a new id). */
int hicr_slot_register(hicr_ctx_t *ctx, void *dev_ptr, uint64_t size, hicr_slot_t *out);

/* Forget a slot (storage untouched).  The caller must have fenced every transfer that
 * names it.  HICR_ERR_INVALID_SLOT on unknown id or double unregister; HICR_ERR_BUSY
 * while a live channel uses it as its ring. */
int hicr_slot_unregister(hicr_ctx_t *ctx, hicr_slot_t slot);

/* Per-slot message counters (host pointers out): `sent` = transfers/tokens whose source
 * was this slot, `recv` = those whose destination was this slot; cumulative since
 * registration (SURVEY.md S8(c) readings 7, 8: the "expected number of incoming and
 * outgoing data transfers" of PAPER.md:375, one message per descriptor / per token).
 * Values are defined immediately after hicr_fence or after a completed channel call. */
int hicr_slot_counters(hicr_ctx_t *ctx, hicr_slot_t slot, uint64_t *sent, uint64_t *recv);

/* ---- memcpy + fence (listing PAPER.md:532-534) ------------------- */

/* Initiate `n` transfers dst[dst_off + i] = src[src_off + i], i < size.
 *
 *   descs            array of n hicr_desc_t.  descs_on_device == 0: host pointer; it is
 *                    validated and consumed before return (the caller may free it).
 *                    descs_on_device != 0: device pointer; it must stay alive and
 *                    unchanged until the next hicr_fence; it is validated on the device.
 *   first_bad        host pointer or NULL; on a host-side validation error receives the
 *                    lowest invalid index.
 *
 * Asynchronous: "The completion of a memory transfer is not guaranteed after the
 * function call returns"; completion and visibility only at hicr_fence.
 * All-or-nothing (reading 10): if any descriptor names an unregistered slot
 * (HICR_ERR_INVALID_SLOT) or a range outside its slot (HICR_ERR_OUT_OF_BOUNDS) the
 * whole batch has no effect and counts nothing; the status is that of the lowest bad
 * index (destination checked before source).  Host-resident tables report it here;
 * device-resident tables report it at hicr_fence.  A zero-size transfer moves nothing
 * and still counts one message (reading 4).  n == 0 is a no-op.
 *
 * Caller contract inside one epoch (= between two fences; reading 5): destination
 * ranges are pairwise disjoint and no destination range overlaps any source range.
 * Sources may overlap; src and dst may be the same slot.  Violations are undefined. */
int hicr_memcpy_batch(hicr_ctx_t *ctx, const hicr_desc_t *descs, uint64_t n, int descs_on_device,
                      uint64_t *first_bad);

/* Block the host until every transfer initiated since the previous fence is complete
 * and visible to the host and to later device work; publish the slot counters; close
 * the epoch ("suspend execution until the expected number of incoming and outgoing data
 * transfers have been completed"; bare fence() as in PAPER.md:534).
 * Returns the first deferred error of the epoch (device-validated batches) or HICR_OK;
 * with nothing outstanding it returns at once.  Batches of the epoch other than the
 * failed one are unaffected. */
int hicr_fence(hicr_ctx_t *ctx);

/* Stream-ordered fence: closes the epoch WITHOUT blocking the host.  Every
 * batch enqueued after it is ordered, on the context's stream, after the completion of every
 * batch enqueued before it, so a later batch may read what an earlier one wrote and the
 * epoch precondition of hicr_memcpy_batch starts afresh.  Nothing is reported here:
 * deferred errors, counters and host visibility come with the next blocking hicr_fence /
 * hicr_fence_expected, whose batch_index then counts batches since the last BLOCKING fence.
 * (The paper's fence is blocking; this is the asynchronous half of it, for
 * chains of dependent epochs such as config 4.) */
int hicr_fence_async(hicr_ctx_t *ctx);

/* Expected-count fence: "suspend execution until the expected number of incoming and outgoing
 * data transfers have been completed".  Blocks the host until slot `slot` has
 * cumulatively sent at least `sent` and received at least `recv` messages (counted since
 * registration, as hicr_slot_counters reports them) AND the transfers counted are complete
 * and visible.  It does not wait for other outstanding batches and does not close the epoch.
 * On return hicr_slot_counters of `slot` reports the values seen.  HICR_ERR_INVALID_SLOT on an
 * unknown slot; HICR_ERR_INVALID_ARG if everything enqueued has completed and the counts are
 * still short (it would block forever); a deferred error of a completed batch is returned as
 * by hicr_fence. */
int hicr_fence_expected(hicr_ctx_t *ctx, hicr_slot_t slot, uint64_t sent, uint64_t recv);

/* ---- replayable chains ("lets config 4 run as one CUDA graph") ---------------
 * Between hicr_graph_begin and hicr_graph_end, hicr_memcpy_batch (device-resident tables only) and
 * hicr_fence_async are RECORDED on the context's stream instead of executed (CUDA stream capture);
 * hicr_graph_launch then enqueues the whole recorded chain with one call, as often as wanted.
 * Every replay validates, bins, copies and counts on the device exactly like the calls it
 * records; completion, counters and deferred errors come with the next blocking hicr_fence,
 * whose batch_index counts the batches since the last blocking fence as usual.  The tables must
 * stay alive and the slot table unchanged from hicr_graph_begin to the last launch, and no
 * hicr_memcpy_batch after the recording may be larger than every batch before it and than
 * max_descs_per_batch (that re-allocates the work queue the recorded launches name):
 * HICR_ERR_INVALID_ARG from hicr_graph_launch otherwise.  While recording, every other call
 * that would enqueue work on the stream returns HICR_ERR_BUSY.  A chain holds at most 64 batches
 * (HICR_ERR_NO_CAPACITY); max_descs_per_batch sizes the work queues up front.  The context must
 * have been created on a stream of its own (HICR_ERR_INVALID_ARG on the legacy default stream,
 * which CUDA cannot capture). */
typedef struct hicr_graph hicr_graph_t;
int hicr_graph_begin(hicr_ctx_t *ctx, uint64_t max_descs_per_batch);
int hicr_graph_end(hicr_ctx_t *ctx, hicr_graph_t **out);
int hicr_graph_launch(hicr_graph_t *g);
int hicr_graph_destroy(hicr_graph_t *g);

/* After hicr_fence returned a deferred error: which batch of that epoch (0-based) and
 * which descriptor index in it was the first bad one.  Host pointers out (may be NULL). */
int hicr_fence_error(hicr_ctx_t *ctx, uint64_t *batch_index, uint64_t *first_bad);

/* ---- memcpy for callers that cannot allocate ---------------------------------
 *
 * hicr_init and hicr_memcpy_batch allocate: the context's tables at start, and the engine's chunk
 * queue again (cudaFree + cudaMalloc, which stall the whole device) whenever a batch is larger
 * than any before it.  That rules the context path out for a process whose HBM was given to its
 * own pool at start-up (a serving engine, a framework's caching allocator: a library's cudaMalloc
 * then fails), and for a step loop with a latency budget that shares the GPU with other streams
 * (they all wait while cudaMalloc / cudaFree run).  This one call is for them.  It needs no
 * context and allocates nothing, on the device or on the host: its work memory -- control words,
 * a per-slot count histogram and the chunk queue -- is one array of about 1 MiB built into the
 * library's device code, which every GPU that runs this library holds until the process exits.
 *
 * One batch, start to end, enqueued on `cuda_stream` (a cudaStream_t of `device`; NULL = the
 * legacy default stream): validate all n descriptors, then -- only if all are valid -- carry out
 * dst[dst_off + i] = src[src_off + i] for each and count one message per descriptor.  It is
 * asynchronous and there is no fence: everything it writes is complete and visible to whatever
 * the caller orders after it on the stream.
 *
 *   d_slots     device pointer, n_slots rows {base, size}; a descriptor's dst_slot / src_slot is an
 *               index into it.  base: device pointer, any alignment.
 *   d_descs     device pointer, n descriptors; unchanged until the call's work is done.
 *   d_counters  device pointer, 2 * n_slots words, in/out: [2 s] += messages whose source was
 *               slot s, [2 s + 1] += messages whose destination was slot s.  The caller zeroes it
 *               once; calls accumulate, as hicr_slot_counters does.
 *   d_result    device pointer, 2 words, out: [0] = HICR_OK, or the status of the lowest bad
 *               descriptor (HICR_ERR_INVALID_SLOT: index >= n_slots; HICR_ERR_OUT_OF_BOUNDS;
 *               destination checked before source), [1] = that descriptor's index.  On an error
 *               nothing was copied and nothing counted, as for hicr_memcpy_batch.
 *
 * Limits, because the work memory cannot grow: n <= HICR_NOALLOC_MAX_DESCS and
 * n_slots <= HICR_NOALLOC_MAX_SLOTS, else HICR_ERR_NO_CAPACITY is returned and nothing is
 * enqueued.  Descriptors above 8 KiB are cut into 128 KiB chunks (size / 128 KiB, rounded up); a
 * batch may hold HICR_NOALLOC_MAX_CHUNKS of them (4 GiB of large transfers).  Only the device sees the
 * sizes, so one chunk too many comes back as d_result[0] = HICR_ERR_NO_CAPACITY with the index
 * of a descriptor that did not fit, and again nothing is copied.
 *
 * Sharing: every call in the process that targets `device` uses the same array, and the array
 * keeps the previous call's contents; each call first clears, in stream order, the part that
 * must start at zero.  Calls on one stream, or otherwise ordered one after the other, are safe.
 * Calls that can run on the GPU at the same time (two streams, no event between them) race on
 * the array: undefined results.
 *
 * The first call for a device looks up where the array sits on that device (once; later calls
 * reuse the address).  Make that first call before any stream capture is in progress.
 *
 * Same caller contract as hicr_memcpy_batch: destination ranges of one batch pairwise disjoint
 * and disjoint from every source range.  Global slots, host-resident tables and profiling belong
 * to the context path only.  Returns HICR_OK once enqueued, HICR_ERR_INVALID_ARG (NULL where
 * needed, device out of range), HICR_ERR_NO_CAPACITY, HICR_ERR_CUDA. */
#define HICR_NOALLOC_MAX_DESCS  65536u
#define HICR_NOALLOC_MAX_SLOTS  1024u
#define HICR_NOALLOC_MAX_CHUNKS 32768u
typedef struct hicr_raw_slot {
    void *base;       /* device pointer */
    uint64_t size;    /* bytes */
} hicr_raw_slot_t;
int hicr_memcpy_batch_noalloc(int device, void *cuda_stream, const hicr_raw_slot_t *d_slots, uint32_t n_slots,
                              const hicr_desc_t *d_descs, uint64_t n, uint64_t *d_counters, int64_t *d_result);

/* ---- Global Memory Slots (S3.1.4) -------------
 *
 * "The communication manager also is in charge of creating and exchanging Global Memory Slots,
 * local memory slots that are made accessible to other HiCR instances and can be used as the
 * source or destination of distributed memcpy operations.  The exchange operation communicates
 * the necessary metadata for remote instances to reach the associated memory slot."
 * (PAPER.md:377).  An INSTANCE here is one context: one process per GPU (or several contexts of
 * one process).  "The exchange of global memory slots is a collective operation: all instances
 * must participate by volunteering zero or more local memory slots.  The operation returns as
 * many global memory slots as the total amount of local memory slots exchanged.  Each of the
 * resulting global memory slots are uniquely identified by a tag and key pair".
 *
 * The library has no transport of its own: the collective is split into its two LOCAL halves,
 * and the caller carries the 256-byte handles between instances over whatever control plane it
 * has (paper_2509_01425_b200/collective.py uses torch.distributed all_gather):
 *   1. every instance calls hicr_global_volunteer once per local slot it volunteers;
 *   2. the handles of ALL instances, in one order all instances agree on, go to
 *      hicr_global_exchange on every instance, which returns one Global Memory Slot id per handle.
 * A global slot id is an ordinary hicr_slot_t of this context: it names the owner's storage --
 * the same address for the owner, a CUDA-IPC / peer mapping of it for every other instance, so a
 * transfer runs in the initiator's copy kernels over NVLink ("the communication
 * manager will use the accelerator-specific network to satisfy the request").  hicr_memcpy_batch
 * takes it as source or destination: Local-to-Local, Local-to-Global (a put) and Global-to-Local
 * (a get) are carried out, a descriptor with two global slots fails the batch with
 * HICR_ERR_ILLEGAL_DIRECTION ("Global-to-Global operations are not permitted").
 * Counters: a message on a global slot counts on the initiator's id like any other, and ALSO at
 * the owner, on the local slot behind it (hicr_global_counters; reading 23). */
#define HICR_GLOBAL_HANDLE_BYTES 256
typedef struct hicr_global_handle {
    unsigned char bytes[HICR_GLOBAL_HANDLE_BYTES];   /* opaque, position-independent, valid on this node */
} hicr_global_handle_t;

/* One line of a global fence's count exchange: what one instance has initiated so far on the
 * global slot (tag, key), cumulative. */
typedef struct hicr_global_count {
    uint64_t tag, key, sent, recv;
} hicr_global_count_t;

/* Plumbing: which instance this context is (default 0 of 1).  Recorded in the handles. */
int hicr_instance_set(hicr_ctx_t *ctx, uint32_t instance, uint32_t n_instances);

/* Local half 1 of the exchange: describe the LOCAL slot `local_slot`, volunteered as (tag, key),
 * in *out (host pointer).  HICR_ERR_INVALID_SLOT on an unknown id, HICR_ERR_INVALID_ARG if the
 * slot is itself a global slot ("volunteering ... local memory slots"). */
int hicr_global_volunteer(hicr_ctx_t *ctx, uint64_t tag, uint64_t key, hicr_slot_t local_slot,
                          hicr_global_handle_t *out);

/* Local half 2: `handles` (host pointer) = the n handles of all instances under `tag`, this
 * context's own included; out_slots (host pointer, n ids) receives the Global Memory Slot of
 * handles[i] at out_slots[i].  All-or-nothing: HICR_ERR_DUPLICATE_KEY if a key occurs twice or
 * (tag, key) exists already in this context, HICR_ERR_INVALID_ARG on a handle that is not one
 * (or of another tag), HICR_ERR_UNSUPPORTED_SPACE if an owner's memory cannot be mapped from this
 * device ("Otherwise, it will be rejected"), HICR_ERR_NO_CAPACITY; then no slot is
 * created.  n == 0 is a valid (empty) exchange.  hicr_slot_unregister drops a global slot again;
 * an owner keeps its storage and its context alive until every instance has dropped the slot. */
int hicr_global_exchange(hicr_ctx_t *ctx, uint64_t tag, const hicr_global_handle_t *handles, uint64_t n,
                         hicr_slot_t *out_slots);

/* The global slot (tag, key) of this context; HICR_ERR_INVALID_SLOT if there is none. */
int hicr_global_lookup(hicr_ctx_t *ctx, uint64_t tag, uint64_t key, hicr_slot_t *out);

/* Global fence, local half 1: hicr_fence (blocks; returns its deferred error, and still reports),
 * then one line per global slot of this context into out[0 .. *n) (host pointers; cap = room in
 * `out`; HICR_ERR_NO_CAPACITY with *n = the number needed if cap is short). */
int hicr_global_fence_begin(hicr_ctx_t *ctx, hicr_global_count_t *out, uint64_t cap, uint64_t *n);

/* Global fence, local half 2: `all` = the lines of ALL instances (any order).  For every global
 * slot this context owns, the expected totals are the sums of its lines; blocks until the
 * owner-side counters on this device have reached them, i.e. until every transfer any instance
 * had initiated on this context's slots when it entered its fence is complete and visible here:
 * "suspend execution until the expected number of incoming and outgoing data transfers have been
 * completed".  HICR_ERR_TIMEOUT after timeout_ms (0 = wait for ever). */
int hicr_global_fence_end(hicr_ctx_t *ctx, const hicr_global_count_t *all, uint64_t n_all, uint32_t timeout_ms);

/* Owner-side totals of a slot of this context (a local slot that was volunteered, or this
 * context's own global id of it): messages of ALL instances that named the global slot as source
 * (sent) / destination (recv).  Defined after hicr_global_fence_end.  Zero for a slot never
 * volunteered; HICR_ERR_INVALID_ARG for a global slot another instance owns. */
int hicr_global_counters(hicr_ctx_t *ctx, hicr_slot_t slot, uint64_t *sent, uint64_t *recv);

/* ---- channels -------------------------------------------------- */

/* SPSC channel over the ring slot: `capacity` tokens of `token_bytes` bytes each; the
 * slot must hold capacity * token_bytes bytes (the pre-allocated circular buffer of
 * PAPER.md:642).  head = tokens ever pushed, tail = tokens ever popped, both 64-bit
 * counters in device memory, 0 at creation.  capacity >= 1, token_bytes >= 1. */
int hicr_channel_create(hicr_ctx_t *ctx, hicr_slot_t ring, uint64_t token_bytes, uint64_t capacity,
                        hicr_channel_t **out);
int hicr_channel_destroy(hicr_channel_t *ch);

/* (head, tail) as of the last completed call on this channel.  Host pointers out. */
int hicr_channel_counters(hicr_channel_t *ch, uint64_t *head, uint64_t *tail);

/* Push min(n_tokens, capacity - (head - tail)) tokens, in order, from slot `src` at
 * byte offset src_off: token j goes to ring position (head + j) mod capacity; head is
 * advanced after the payload is visible ("the producer knows where to push the next
 * message, as long as the buffer has not filled up").  *n_pushed (host
 * pointer) receives the count; 0 with n_tokens > 0 = full.  The source range of
 * n_tokens * token_bytes bytes must lie inside `src`.  Complete on return.  Counts one
 * message per token: sent(src), recv(ring).  The k decision is taken on the device from
 * the device-resident counters. */
int hicr_channel_push(hicr_channel_t *ch, hicr_slot_t src, uint64_t src_off, uint64_t n_tokens,
                      uint64_t *n_pushed);

/* Pop k = min(max_tokens, head - tail) tokens in FIFO order into slot `dst` at dst_off:
 * token j comes from ring position (tail + j) mod capacity; tail is advanced once per
 * call after the reads are done ("the consumer notifies that a message has been
 * consumed").  *n_popped receives k; 0 = empty.  The range of
 * k * token_bytes bytes must lie inside `dst` (else HICR_ERR_OUT_OF_BOUNDS, no effect).
 * Complete on return.  Counts sent(ring), recv(dst). */
int hicr_channel_pop(hicr_channel_t *ch, hicr_slot_t dst, uint64_t dst_off, uint64_t max_tokens,
                     uint64_t *n_popped);

/* Device-resident SPSC run: one kernel in which a producer CTA performs, for
 * i < n_batches, a blocking push of batch_tokens[i] tokens (waiting on the device for
 * room) from `src` (consecutive tokens starting at src_off) while a consumer CTA
 * concurrently pops whatever is available into `dst` (consecutive from dst_off) until
 * all sum(batch_tokens) tokens are through.  batch_tokens: host pointer, consumed
 * before return.  Blocks until done.  On return head and tail have advanced by the sum
 * and the counters by one message per token, exactly as the equivalent sequence of
 * hicr_channel_push / hicr_channel_pop calls would leave them.  Requires an empty ring
 * (head == tail) at entry. */
int hicr_channel_stream(hicr_channel_t *ch, hicr_slot_t src, uint64_t src_off, hicr_slot_t dst,
                        uint64_t dst_off, const uint64_t *batch_tokens, uint64_t n_batches);

/* Non-locking MPSC ("dedicated buffers per producer"): `producers` SPSC
 * rings, rings[p] the ring slot of producer p (host pointer to `producers` ids). */
int hicr_mpsc_create(hicr_ctx_t *ctx, uint32_t producers, const hicr_slot_t *rings, uint64_t token_bytes,
                     uint64_t capacity, hicr_mpsc_t **out);
int hicr_mpsc_destroy(hicr_mpsc_t *m);
int hicr_mpsc_counters(hicr_mpsc_t *m, uint32_t producer, uint64_t *head, uint64_t *tail);

/* Device-resident MPSC run: producer p pushes tokens_per_producer tokens from slot src_slots[p],
 * consecutively from byte offset src_offs[p], into its own ring in batches of at most max_batch
 * tokens, waiting for room on the device; the single logical consumer pops what is available
 * into dst_slots[p], consecutively from dst_offs[p].  Per-producer FIFO.  head_p and tail_p
 * continue from where the previous run left them (token i of the ring's lifetime sits at ring
 * position i mod capacity).  src_slots / dst_slots: host pointers to
 * `producers` ids; src_offs / dst_offs: host pointers to `producers` byte offsets, or NULL for
 * all zero.  Requires head_p == tail_p at entry.  Blocks until done; counters as for
 * hicr_channel_stream. */
int hicr_mpsc_stream(hicr_mpsc_t *m, const hicr_slot_t *src_slots, const uint64_t *src_offs,
                     const hicr_slot_t *dst_slots, const uint64_t *dst_offs, uint64_t tokens_per_producer,
                     uint64_t max_batch);

/* Device-resident LOCKING MPSC run ("locking, where a collective exclusive
 * access guarantees a shared channel does not overflow"): `producers` producer CTAs push
 * tokens_per_producer tokens each, from src_slots[p] (offset 0), into the ONE ring of the
 * SPSC channel `ch`, in batches of at most max_batch tokens; a single consumer CTA pops them
 * into `dst`, consecutively from dst_off, in the order they entered the ring.  The
 * exclusive access is an atomic reservation of ring positions that succeeds only while the
 * positions are free, followed by a commit in reservation order.  The interleaving of
 * producers in `dst` is not defined; what is: each producer's tokens appear in its own
 * order (per-producer FIFO), every token exactly once, head = tail advanced by
 * producers * tokens_per_producer, one message per token on every slot.  Requires an empty
 * ring at entry and all producers + 1 CTAs co-resident (HICR_ERR_NO_CAPACITY otherwise).
 * src_slots: host pointer to `producers` ids.  Blocks until done. */
int hicr_mpsc_locking_stream(hicr_channel_t *ch, uint32_t producers, const hicr_slot_t *src_slots, hicr_slot_t dst,
                             uint64_t dst_off, uint64_t tokens_per_producer, uint64_t max_batch);

/* ---- measurement hooks (plumbing) -------------------------------------------------- */

/* Kernel launches issued by this context since hicr_init (host pointer out). */
int hicr_launch_count(hicr_ctx_t *ctx, uint64_t *launches);

/* With profiling on, every hicr_memcpy_batch records CUDA events around its engine kernel
 * on the context's stream.  hicr_profile_read (only right after a fence) returns, for the
 * LAST batch, in milliseconds: [0] the validation/binning phase up to the grid barrier and
 * [1] the copy phase, both from the device's %globaltimer stamps in the completion record,
 * [2] their sum, [3] the whole kernel from the CUDA events.  ms: host pointer to 4 floats. */
int hicr_profile_enable(hicr_ctx_t *ctx, int on);
int hicr_profile_read(hicr_ctx_t *ctx, float *ms);

#ifdef __cplusplus
}
#endif
#endif /* HICR_H */
