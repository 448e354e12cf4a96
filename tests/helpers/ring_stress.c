/* Test helper: two host threads hammer cc_submit on ONE context at the same time (SURVEY.md section 5 row 2,
 * "2-thread stress test"; the ring is single-producer).  The library must refuse the thread that
 * finds the other one inside cc_submit (CC_ERR_INVALID, -1) and must neither lose nor duplicate a task.
 * Plain C + pthreads; the cc_submit pointer is passed in, nothing of the product is linked or included. */
#include <pthread.h>
#include <stdint.h>
#include <string.h>

typedef struct { uint32_t kind, region_id, flags, version; uint64_t seq, epoch, arg0, arg1, arg2, arg3; } task64;
typedef int32_t (*submit_fn)(void*, const void*, uint64_t*);

struct side {
    submit_fn submit; void* ctx; uint32_t n, tag; uint64_t* seqs;
    uint64_t refused, full; int32_t err; pthread_barrier_t* bar;
};

static void* producer(void* p) {
    struct side* s = (struct side*)p;
    pthread_barrier_wait(s->bar);
    for (uint32_t i = 0; i < s->n; i++) {
        task64 t;
        memset(&t, 0, sizeof t);                            /* kind 0 = CC_TASK_NOP */
        t.epoch = ((uint64_t)s->tag << 32) | i;             /* echoed into the completion record */
        for (;;) {
            uint64_t seq = ~0ull;
            const int32_t rc = s->submit(s->ctx, &t, &seq);
            if (rc == 0) { s->seqs[i] = seq; break; }
            if (rc == -1) s->refused++;                     /* the other producer was inside */
            else if (rc == -6) s->full++;                   /* CC_ERR_RING_FULL: the worker has to catch up */
            else { s->err = rc; return 0; }
        }
    }
    return 0;
}

/* counters: refused_a, refused_b, full_a, full_b.  Returns 0, or the first unexpected status. */
int32_t ring_stress(void* submit, void* ctx, uint32_t n, uint64_t* seqs_a, uint64_t* seqs_b, uint64_t* counters) {
    pthread_barrier_t bar;
    pthread_barrier_init(&bar, 0, 2);
    struct side a = {(submit_fn)submit, ctx, n, 1, seqs_a, 0, 0, 0, &bar};
    struct side b = {(submit_fn)submit, ctx, n, 2, seqs_b, 0, 0, 0, &bar};
    pthread_t ta, tb;
    pthread_create(&ta, 0, producer, &a);
    pthread_create(&tb, 0, producer, &b);
    pthread_join(ta, 0);
    pthread_join(tb, 0);
    pthread_barrier_destroy(&bar);
    counters[0] = a.refused; counters[1] = b.refused; counters[2] = a.full; counters[3] = b.full;
    return a.err ? a.err : b.err;
}
