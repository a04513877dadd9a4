/*
 * hicr_oracle.c -- CPU ORACLE for the HiCR memory-slot memcpy / fence / channel path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_2509_01425_b200/csrc/ and includes nothing from include/.
 *
 * It is the plain definition of what the path computes, written as single-threaded
 * byte loops in the paper's order and notation (PAPER.md = arxiv 2509.01425):
 *
 *   - Local Memory Slot: "the minimum information required to describe a segment of
 *     memory (e.g., size, starting address)"                  PAPER.md:364  (S3.1.3)
 *   - manual registration of an existing allocation            PAPER.md:368  (S3.1.3)
 *   - memcpy(dst slot, dst offset, src slot, src offset, size); initiated if supported,
 *     "Otherwise, it will be rejected"                         PAPER.md:373, listing :532
 *   - completion only at the fence: "suspend execution until the expected number of
 *     incoming and outgoing data transfers have been completed" PAPER.md:375, listing :534
 *   - Channels: pre-allocated circular buffer at the consumer; the producer pushes "as
 *     long as the buffer has not filled up"; the consumer "notifies that a message has
 *     been consumed"                                            PAPER.md:642  (S4.3)
 *   - MPSC non-locking: "dedicated buffers per producer"        PAPER.md:644  (S4.3)
 *
 * Readings of points where the paper is silent are those of SURVEY.md S8(c) and are
 * listed in DESIGN.md ("Readings").  Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   oracle_memcpy_batch   pinned: exhaustive brute force vs the closed form, libc memmove,
 *                         printed examples (tests/golden/), permutation invariance,
 *                         the paper's broadcast listing.
 *   oracle_fence/counters pinned by closed-form descriptor counts and config 1's value
 *                         256; the PER-SLOT ATTRIBUTION itself is a reading (S8(c) pt 7):
 *                         "parity unpinned" by the paper for that attribution.
 *   oracle_channel_*      pinned: differential test against a queue of byte strings,
 *                         invariants 0 <= head-tail <= C, capacity-1 and capacity-4
 *                         printed examples.
 *   partial-push rule, zero-size rule, all-or-nothing errors: "parity unpinned" by the
 *                         paper (SURVEY S8(c) pts 4, 10, 12); fixed by unit tests.
 *
 * Global Memory Slots (S3.1.4): several oracle
 * contexts stand for several HiCR instances in one process.  A Global Memory Slot is "a local
 * memory slot ... made accessible to other HiCR instances": here a slot of
 * kind GLOBAL in the table of every instance, over the storage of the volunteered local slot
 * of its owner.  The collective exchange itself (who volunteers what under which tag and key)
 * is oracle/world.py; this file holds the three legal directions -- "Global-to-Global
 * operations are not permitted" -- and the counters.
 *   oracle_slot_register_global / direction rule  pinned: the four slot-kind pairs of
 *                         SPEC.md:78-84, the 2-instance put / get examples,
 *                         a randomized copy graph against numpy slicing.
 *   global counters (every message naming a global slot also counts at its owner, reading
 *                         23 of DESIGN.md): "parity unpinned" by the paper; pinned to the
 *                         closed form sum over instances of their own per-slot counts.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* status codes (values fixed by DESIGN.md "Status codes"; typed here independently) */
enum {
    ORC_OK = 0,
    ORC_ERR_INVALID_ARG = -1,
    ORC_ERR_INVALID_SLOT = -2,
    ORC_ERR_OUT_OF_BOUNDS = -3,
    ORC_ERR_NO_CAPACITY = -5,
    ORC_ERR_ILLEGAL_DIRECTION = -8   /* "Global-to-Global operations are not permitted" */
};

struct orc_ctx_s;

typedef struct {
    uint8_t *base;   /* starting address */
    uint64_t size;   /* size in bytes */
    uint64_t sent;   /* messages sent from this slot, cumulative (reading 7) */
    uint64_t recv;   /* messages received into this slot, cumulative (reading 7) */
    int valid;
    /* Global Memory Slot: the local slot `owner_slot` of instance `owner`, seen
     * from this instance.  g_sent / g_recv of THAT local slot count the messages of all
     * instances that named the global slot as source / destination (reading 23). */
    int global;
    struct orc_ctx_s *owner;
    uint32_t owner_slot;
    uint64_t g_sent, g_recv;
} orc_slot;

/* field order = the paper's call: dst, dst offset, src, src offset, size */
typedef struct {
    uint32_t dst_slot;
    uint32_t src_slot;
    uint64_t dst_off;
    uint64_t src_off;
    uint64_t size;
} orc_desc;

typedef struct {
    uint32_t src_slot;
    uint32_t dst_slot;
} orc_pending;

typedef struct {
    uint32_t ring_slot;
    uint64_t T;      /* token size in bytes */
    uint64_t C;      /* capacity in tokens  */
    uint64_t head;   /* tokens ever pushed (reading 11) */
    uint64_t tail;   /* tokens ever popped (reading 11) */
    int valid;
} orc_channel;

typedef struct orc_ctx_s {
    orc_slot *slots;
    uint32_t n_slots, cap_slots;
    orc_pending *pending;
    uint64_t n_pending, cap_pending;
    orc_channel *channels;
    uint32_t n_channels, cap_channels;
} orc_ctx;

orc_ctx *oracle_new(void) { return (orc_ctx *)calloc(1, sizeof(orc_ctx)); }

void oracle_free(orc_ctx *o)
{
    if (!o) return;
    free(o->slots);
    free(o->pending);
    free(o->channels);
    free(o);
}

/* register(ptr, size): append a slot with sent = recv = 0.  Size 0 allowed. */
int oracle_slot_register(orc_ctx *o, uint8_t *ptr, uint64_t size, uint32_t *out)
{
    if (!o || !out || (!ptr && size)) return ORC_ERR_INVALID_ARG;
    if (o->n_slots == o->cap_slots) {
        uint32_t nc = o->cap_slots ? o->cap_slots * 2 : 16;
        orc_slot *ns = (orc_slot *)realloc(o->slots, (size_t)nc * sizeof(orc_slot));
        if (!ns) return ORC_ERR_NO_CAPACITY;
        o->slots = ns;
        o->cap_slots = nc;
    }
    orc_slot *s = &o->slots[o->n_slots];
    s->base = ptr;
    s->size = size;
    s->sent = 0;
    s->recv = 0;
    s->valid = 1;
    s->global = 0;
    s->owner = NULL;
    s->owner_slot = 0;
    s->g_sent = 0;
    s->g_recv = 0;
    *out = o->n_slots++;
    return ORC_OK;
}

/* One instance's view of a Global Memory Slot: the storage of local slot `owner_slot` of
 * instance `owner` (which may be `o` itself), "made accessible to other HiCR instances"
 * (PAPER.md:377).  Same size and starting address as the local slot behind it. */
int oracle_slot_register_global(orc_ctx *o, orc_ctx *owner, uint32_t owner_slot, uint32_t *out)
{
    if (!o || !owner || !out) return ORC_ERR_INVALID_ARG;
    if (owner_slot >= owner->n_slots || !owner->slots[owner_slot].valid) return ORC_ERR_INVALID_SLOT;
    if (owner->slots[owner_slot].global) return ORC_ERR_INVALID_ARG;   /* only local slots are volunteered */
    {
        /* (o == owner: the table may move when it grows, so take the values first) */
        uint8_t *base = owner->slots[owner_slot].base;
        uint64_t size = owner->slots[owner_slot].size;
        int rc = oracle_slot_register(o, base, size, out);
        if (rc != ORC_OK) return rc;
    }
    o->slots[*out].global = 1;
    o->slots[*out].owner = owner;
    o->slots[*out].owner_slot = owner_slot;
    return ORC_OK;
}

/* 1 if `slot` is this instance's view of a Global Memory Slot, 0 if it is a Local Memory Slot. */
int oracle_slot_is_global(orc_ctx *o, uint32_t slot)
{
    if (!o) return ORC_ERR_INVALID_ARG;
    if (slot >= o->n_slots || !o->slots[slot].valid) return ORC_ERR_INVALID_SLOT;
    return o->slots[slot].global;
}

/* Messages of ALL instances that named the Global Memory Slot behind local slot `slot` of
 * this instance as source (sent) / destination (recv); complete once every instance has
 * fenced (reading 23). */
int oracle_slot_global_counters(orc_ctx *o, uint32_t slot, uint64_t *sent, uint64_t *recv)
{
    if (!o || !sent || !recv) return ORC_ERR_INVALID_ARG;
    if (slot >= o->n_slots || !o->slots[slot].valid) return ORC_ERR_INVALID_SLOT;
    *sent = o->slots[slot].g_sent;
    *recv = o->slots[slot].g_recv;
    return ORC_OK;
}

int oracle_slot_unregister(orc_ctx *o, uint32_t slot)
{
    if (!o) return ORC_ERR_INVALID_ARG;
    if (slot >= o->n_slots || !o->slots[slot].valid) return ORC_ERR_INVALID_SLOT;
    o->slots[slot].valid = 0;
    return ORC_OK;
}

int oracle_slot_counters(orc_ctx *o, uint32_t slot, uint64_t *sent, uint64_t *recv)
{
    if (!o || !sent || !recv) return ORC_ERR_INVALID_ARG;
    if (slot >= o->n_slots || !o->slots[slot].valid) return ORC_ERR_INVALID_SLOT;
    *sent = o->slots[slot].sent;
    *recv = o->slots[slot].recv;
    return ORC_OK;
}

/* overflow-safe form of "offset + size <= slot size" (SURVEY S8(c) definition) */
static int range_ok(const orc_slot *s, uint64_t off, uint64_t size)
{
    if (off > s->size) return 0;
    if (size > s->size - off) return 0;
    return 1;
}

static int check_range(const orc_ctx *o, uint32_t slot, uint64_t off, uint64_t size)
{
    if (slot >= o->n_slots || !o->slots[slot].valid) return ORC_ERR_INVALID_SLOT;
    if (!range_ok(&o->slots[slot], off, size)) return ORC_ERR_OUT_OF_BOUNDS;
    return ORC_OK;
}

/* dst[dst_off+i] = src[src_off+i], i < size: the byte loop that defines a transfer
 * (PAPER.md:373).  When both ranges lie in the same slot and overlap, the copy goes
 * through a temporary, i.e. it reads the bytes "at initiation time". */
static void copy_bytes(uint8_t *dst, const uint8_t *src, uint64_t size)
{
    uint64_t i;
    if (size == 0) return;
    if ((dst < src + size) && (src < dst + size) && dst != src) {
        uint8_t *tmp = (uint8_t *)malloc((size_t)size);
        for (i = 0; i < size; i++) tmp[i] = src[i];
        for (i = 0; i < size; i++) dst[i] = tmp[i];
        free(tmp);
        return;
    }
    for (i = 0; i < size; i++) dst[i] = src[i];
}

static int push_pending(orc_ctx *o, uint32_t src_slot, uint32_t dst_slot)
{
    if (o->n_pending == o->cap_pending) {
        uint64_t nc = o->cap_pending ? o->cap_pending * 2 : 1024;
        orc_pending *np = (orc_pending *)realloc(o->pending, (size_t)nc * sizeof(orc_pending));
        if (!np) return ORC_ERR_NO_CAPACITY;
        o->pending = np;
        o->cap_pending = nc;
    }
    o->pending[o->n_pending].src_slot = src_slot;
    o->pending[o->n_pending].dst_slot = dst_slot;
    o->n_pending++;
    return ORC_OK;
}

/* memcpy_batch: check every descriptor first; any failure rejects the whole batch with
 * no effect ("Otherwise, it will be rejected"; all-or-nothing = reading 10);
 * otherwise apply the descriptors in index order and append them to the pending list. */
int oracle_memcpy_batch(orc_ctx *o, const orc_desc *d, uint64_t n, uint64_t *first_bad)
{
    uint64_t k;
    if (!o || (!d && n)) return ORC_ERR_INVALID_ARG;
    for (k = 0; k < n; k++) {
        int rc = check_range(o, d[k].dst_slot, d[k].dst_off, d[k].size);
        if (rc == ORC_OK) rc = check_range(o, d[k].src_slot, d[k].src_off, d[k].size);
        /* Local-to-Local, Local-to-Global and Global-to-Local only */
        if (rc == ORC_OK && o->slots[d[k].dst_slot].global && o->slots[d[k].src_slot].global)
            rc = ORC_ERR_ILLEGAL_DIRECTION;
        if (rc != ORC_OK) {
            if (first_bad) *first_bad = k;
            return rc;
        }
    }
    for (k = 0; k < n; k++) {
        orc_slot *ds = &o->slots[d[k].dst_slot];
        orc_slot *ss = &o->slots[d[k].src_slot];
        copy_bytes(ds->base + d[k].dst_off, ss->base + d[k].src_off, d[k].size);
        int rc = push_pending(o, d[k].src_slot, d[k].dst_slot);
        if (rc != ORC_OK) return rc;
    }
    return ORC_OK;
}

/* fence: every pending transfer is complete (they were applied eagerly); count one
 * outgoing message on its source slot and one incoming message on its destination slot
 * ("incoming and outgoing data transfers"; readings 4, 7, 8), clear pending. */
int oracle_fence(orc_ctx *o)
{
    uint64_t k;
    if (!o) return ORC_ERR_INVALID_ARG;
    for (k = 0; k < o->n_pending; k++) {
        orc_slot *ss = &o->slots[o->pending[k].src_slot];
        orc_slot *ds = &o->slots[o->pending[k].dst_slot];
        ss->sent += 1;
        ds->recv += 1;
        /* a global slot's message also counts at its owner, on the local slot behind it */
        if (ss->global) ss->owner->slots[ss->owner_slot].g_sent += 1;
        if (ds->global) ds->owner->slots[ds->owner_slot].g_recv += 1;
    }
    o->n_pending = 0;
    return ORC_OK;
}

uint64_t oracle_pending(orc_ctx *o) { return o ? o->n_pending : 0; }

/* ------------------------------------------------------------------ channels (S4.3) */

int oracle_channel_create(orc_ctx *o, uint32_t ring_slot, uint64_t T, uint64_t C, uint32_t *out)
{
    if (!o || !out) return ORC_ERR_INVALID_ARG;
    if (T == 0 || C == 0) return ORC_ERR_INVALID_ARG;          /* capacity >= 1 */
    if (ring_slot >= o->n_slots || !o->slots[ring_slot].valid) return ORC_ERR_INVALID_SLOT;
    if (C > UINT64_MAX / T) return ORC_ERR_OUT_OF_BOUNDS;
    if (C * T > o->slots[ring_slot].size) return ORC_ERR_OUT_OF_BOUNDS;
    if (o->n_channels == o->cap_channels) {
        uint32_t nc = o->cap_channels ? o->cap_channels * 2 : 16;
        orc_channel *nch = (orc_channel *)realloc(o->channels, (size_t)nc * sizeof(orc_channel));
        if (!nch) return ORC_ERR_NO_CAPACITY;
        o->channels = nch;
        o->cap_channels = nc;
    }
    orc_channel *c = &o->channels[o->n_channels];
    c->ring_slot = ring_slot;
    c->T = T;
    c->C = C;
    c->head = 0;
    c->tail = 0;
    c->valid = 1;
    *out = o->n_channels++;
    return ORC_OK;
}

int oracle_channel_counters(orc_ctx *o, uint32_t ch, uint64_t *head, uint64_t *tail)
{
    if (!o || !head || !tail || ch >= o->n_channels) return ORC_ERR_INVALID_ARG;
    *head = o->channels[ch].head;
    *tail = o->channels[ch].tail;
    return ORC_OK;
}

/* push: k = min(n, C - (head - tail)) tokens, token j of the call goes to ring position
 * (head + j) mod C; then head += k; one message per token on the counters (reading 15).
 * "the producer knows where to push the next message, as long as the buffer has not
 * filled up". */
int oracle_channel_push(orc_ctx *o, uint32_t ch, uint32_t src, uint64_t src_off, uint64_t n,
                        uint64_t *n_pushed)
{
    uint64_t j, i, k, room;
    if (!o || !n_pushed || ch >= o->n_channels) return ORC_ERR_INVALID_ARG;
    orc_channel *c = &o->channels[ch];
    if (src >= o->n_slots || !o->slots[src].valid) return ORC_ERR_INVALID_SLOT;
    if (n > UINT64_MAX / c->T) return ORC_ERR_OUT_OF_BOUNDS;
    if (!range_ok(&o->slots[src], src_off, n * c->T)) return ORC_ERR_OUT_OF_BOUNDS;
    room = c->C - (c->head - c->tail);
    k = n < room ? n : room;
    {
        const uint8_t *s = o->slots[src].base + src_off;
        uint8_t *ring = o->slots[c->ring_slot].base;
        for (j = 0; j < k; j++) {
            uint64_t pos = (c->head + j) % c->C;
            for (i = 0; i < c->T; i++) ring[pos * c->T + i] = s[j * c->T + i];
        }
    }
    c->head += k;
    o->slots[src].sent += k;
    o->slots[c->ring_slot].recv += k;
    *n_pushed = k;
    return ORC_OK;
}

/* pop: k = min(max, head - tail) tokens, token j of the call comes from ring position
 * (tail + j) mod C; then tail += k ("the consumer notifies that a message has been
 * consumed"; once per call = reading 14). */
int oracle_channel_pop(orc_ctx *o, uint32_t ch, uint32_t dst, uint64_t dst_off, uint64_t max_n,
                       uint64_t *n_popped)
{
    uint64_t j, i, k, depth;
    if (!o || !n_popped || ch >= o->n_channels) return ORC_ERR_INVALID_ARG;
    orc_channel *c = &o->channels[ch];
    if (dst >= o->n_slots || !o->slots[dst].valid) return ORC_ERR_INVALID_SLOT;
    depth = c->head - c->tail;
    k = max_n < depth ? max_n : depth;
    if (k > UINT64_MAX / c->T) return ORC_ERR_OUT_OF_BOUNDS;
    if (!range_ok(&o->slots[dst], dst_off, k * c->T)) return ORC_ERR_OUT_OF_BOUNDS;
    {
        uint8_t *d = o->slots[dst].base + dst_off;
        const uint8_t *ring = o->slots[c->ring_slot].base;
        for (j = 0; j < k; j++) {
            uint64_t pos = (c->tail + j) % c->C;
            for (i = 0; i < c->T; i++) d[j * c->T + i] = ring[pos * c->T + i];
        }
    }
    c->tail += k;
    o->slots[c->ring_slot].sent += k;
    o->slots[dst].recv += k;
    *n_popped = k;
    return ORC_OK;
}
