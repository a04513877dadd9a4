/*
 * parallel_memcpy.c -- the STRONGER CPU BASELINE of SURVEY.md S8(d): the descriptor loop of
 * the memcpy path with libc memcpy, descriptors spread over all the host cores the process
 * may use.  TIMING BASELINE ONLY (bench.py's cpu_baseline_parallel): it is not the oracle,
 * proves nothing about parity and validates nothing (it is handed descriptor sets the
 * oracle has accepted).  tests/test_oracle_memcpy.py checks its image against the oracle's.
 * Shares no code with the CUDA path; includes nothing from include/.
 *
 * "dst[dst_off + i] = src[src_off + i], i < size" (field order of the listing
 * PAPER.md:532) under the epoch precondition of SURVEY.md S8(c) point 5 (destinations
 * pairwise disjoint, none overlapping a source), which makes the descriptors independent.
 */
#include <pthread.h>
#include <stdatomic.h>
#include <stdint.h>
#include <string.h>

typedef struct {
    uint32_t dst_slot, src_slot;
    uint64_t dst_off, src_off, size;
} pm_desc;

typedef struct {
    uint8_t *const *bases;
    const pm_desc *d;
    uint64_t n;
    atomic_ullong next;
} pm_job;

enum { PM_GRAIN = 64 };   /* descriptors per claim */

static void *pm_worker(void *arg)
{
    pm_job *j = (pm_job *)arg;
    for (;;) {
        const uint64_t i0 = atomic_fetch_add_explicit(&j->next, PM_GRAIN, memory_order_relaxed);
        if (i0 >= j->n) return 0;
        const uint64_t i1 = i0 + PM_GRAIN < j->n ? i0 + PM_GRAIN : j->n;
        for (uint64_t i = i0; i < i1; i++) {
            const pm_desc *d = &j->d[i];
            memcpy(j->bases[d->dst_slot] + d->dst_off, j->bases[d->src_slot] + d->src_off, d->size);
        }
    }
}

/* bases[s] = starting address of slot s.  Returns 0, or -1 if a thread could not be started. */
int parallel_memcpy_batch(uint8_t *const *bases, const pm_desc *d, uint64_t n, int threads)
{
    pm_job j;
    pthread_t t[256];
    int started = 0, rc = 0;
    j.bases = bases;
    j.d = d;
    j.n = n;
    atomic_init(&j.next, 0);
    if (threads > 256) threads = 256;
    for (int k = 1; k < threads; k++) {
        if (pthread_create(&t[started], 0, pm_worker, &j) != 0) {
            rc = -1;
            break;
        }
        started++;
    }
    pm_worker(&j);
    for (int k = 0; k < started; k++) pthread_join(t[k], 0);
    return rc;
}
