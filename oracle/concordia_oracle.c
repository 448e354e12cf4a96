/*
 * concordia_oracle.c -- CPU ORACLE for the Concordia delta-checkpoint hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the slow, plain, obviously-correct
 * definition that the CUDA path (paper_2606_23521_b200/csrc) is checked against.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call it.  It shares no code, header, table
 * or constant generator with the CUDA path; the on-disk record format constants
 * are re-typed here from DESIGN.md / SURVEY.md section 8c.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md, text of arxiv 2606.23521):
 *   - dirty discovery: "comparing against GPU-resident shadow copies at 4 KB page
 *     granularity" (section 3.3; L261, section 4.2 stage 1)  -> memcmp per page
 *   - record: "an AOF record containing the epoch, region ID, dirty page
 *     descriptors, payload offsets, and a checksum" (L219); "region ID, version,
 *     dirty page list, payload, and commit marker" (L85, section 2.3)
 *   - discipline: "write record header, write dirty payloads, write commit
 *     marker, then publish the epoch. Recovery ignores any suffix without a commit
 *     marker." (L221)
 *   - shadow update: "opaque-region shadows are overwritten with current contents
 *     for the next delta" (L264, stage 4)
 *   - restore: "fn.apply(aof_read(desc.epoch))" (L156-158); "replays the latest
 *     base snapshot and committed AOF suffix" (L227)
 * The byte-level format (the paper names the fields but not their widths) is the
 * reading fixed in DESIGN.md "Readings of the paper":
 *   page record  = 16-byte little-endian header {u32 region_id, u32 page_idx,
 *                  u32 len, u32 crc32c(payload)} followed by len payload bytes
 *   commit record= header {0xFFFFFFFF, 0xFFFFFFFF, 16, crc32c(payload)} followed by
 *                  16-byte payload {u64 epoch, u32 region_id, u32 k}
 * CRC32C = Castagnoli, reflected polynomial 0x82F63B78, init 0xFFFFFFFF, final
 * XOR 0xFFFFFFFF (BASELINE.json north_star; check value 0xE3069283 on "123456789").
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): CRC check value and the iSCSI
 * 32-byte vectors, the SSE4.2 crc32 instruction, the two worked examples of
 * SURVEY.md section 8c (tests/golden/), closed-form log sizes, brute force over all
 * dirty subsets of tiny regions, round-trip / idempotence / truncation sweeps.
 *
 * No blocking, fusion, SIMD or threading: every function is the definition
 * written out.  (orc_scan_mt at the bottom only partitions the page range of
 * the same memcmp loop over pthreads, for the "all host cores" baseline line.)
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#include <stdlib.h>
#include <pthread.h>

#define ORC_OK 0
#define ORC_ERR_INVALID (-1)
#define ORC_ERR_LOG_FULL (-4)
#define ORC_ERR_CORRUPT (-5)

#define ORC_COMMIT_ID 0xFFFFFFFFu
#define ORC_HDR 16u
#define ORC_COMMIT_BYTES 32u

/* ---------------------------------------------------------------- CRC32C --- */

/* Bit-at-a-time definition: reflected CRC, polynomial 0x82F63B78. */
uint32_t orc_crc32c_bitwise(const uint8_t *p, uint64_t n) {
    uint32_t crc = 0xFFFFFFFFu;
    for (uint64_t i = 0; i < n; i++) {
        crc ^= p[i];
        for (int b = 0; b < 8; b++)
            crc = (crc & 1u) ? (crc >> 1) ^ 0x82F63B78u : (crc >> 1);
    }
    return crc ^ 0xFFFFFFFFu;
}

static uint32_t orc_table[256];
static int orc_table_ready = 0;

static void orc_make_table(void) {
    for (uint32_t i = 0; i < 256; i++) {
        uint32_t c = i;
        for (int b = 0; b < 8; b++)
            c = (c & 1u) ? (c >> 1) ^ 0x82F63B78u : (c >> 1);
        orc_table[i] = c;
    }
    orc_table_ready = 1;
}

/* Byte-at-a-time, 256-entry table (the textbook Sarwate loop). */
uint32_t orc_crc32c(const uint8_t *p, uint64_t n) {
    if (!orc_table_ready) orc_make_table();
    uint32_t crc = 0xFFFFFFFFu;
    for (uint64_t i = 0; i < n; i++)
        crc = orc_table[(crc ^ p[i]) & 0xFFu] ^ (crc >> 8);
    return crc ^ 0xFFFFFFFFu;
}

/* ------------------------------------------------------- little-endian io --- */

static void put_u32(uint8_t *p, uint32_t v) {
    p[0] = (uint8_t)(v); p[1] = (uint8_t)(v >> 8); p[2] = (uint8_t)(v >> 16); p[3] = (uint8_t)(v >> 24);
}
static void put_u64(uint8_t *p, uint64_t v) {
    put_u32(p, (uint32_t)v); put_u32(p + 4, (uint32_t)(v >> 32));
}
static uint32_t get_u32(const uint8_t *p) {
    return (uint32_t)p[0] | ((uint32_t)p[1] << 8) | ((uint32_t)p[2] << 16) | ((uint32_t)p[3] << 24);
}

/* ------------------------------------------------------------------ scan --- */

static uint64_t page_len(uint64_t N, uint64_t P, uint64_t p) {
    uint64_t start = p * P;
    uint64_t rest = N - start;
    return rest < P ? rest : P;
}

/* Step 1-2 of the checkpoint oracle:
 * dirty[p] = memcmp(cur + p*P, shadow + p*P, len_p) != 0.  Returns k. */
uint64_t orc_scan(const uint8_t *cur, const uint8_t *shadow, uint64_t N, uint64_t P, uint8_t *dirty) {
    uint64_t n_pages = (N + P - 1) / P;
    uint64_t k = 0;
    for (uint64_t p = 0; p < n_pages; p++) {
        uint64_t len = page_len(N, P, p);
        int d = memcmp(cur + p * P, shadow + p * P, len) != 0;
        dirty[p] = (uint8_t)d;
        k += (uint64_t)d;
    }
    return k;
}

/* ------------------------------------------------------------ checkpoint --- */

/* Full checkpoint oracle, steps 1-9 of SURVEY.md 8c.
 *   cur, shadow : N bytes each; shadow is updated in place for dirty pages
 *   log, C, *W  : append-only log buffer, its capacity, running write offset
 *   D_out       : room for n_pages u32 (ascending dirty list), may be NULL
 *   *k_out      : number of dirty pages;  *bytes_out : bytes appended
 * Returns ORC_OK, ORC_ERR_LOG_FULL (nothing written, shadow untouched) or
 * ORC_ERR_INVALID. */
int32_t orc_checkpoint(const uint8_t *cur, uint8_t *shadow, uint64_t N, uint64_t P,
                       uint32_t region_id, uint64_t epoch,
                       uint8_t *log, uint64_t C, uint64_t *W,
                       uint32_t *D_out, uint64_t *k_out, uint64_t *bytes_out) {
    if (P == 0 || N == 0 || region_id == 0 || region_id == ORC_COMMIT_ID) return ORC_ERR_INVALID;
    uint64_t n_pages = (N + P - 1) / P;
    if (n_pages > 0xFFFFFFFEull) return ORC_ERR_INVALID;

    /* steps 2-3: dirty set, ascending */
    uint8_t *dirty = (uint8_t *)malloc(n_pages);
    if (!dirty) return ORC_ERR_INVALID;
    uint64_t k = orc_scan(cur, shadow, N, P, dirty);
    *k_out = k;
    *bytes_out = 0;
    if (D_out) {
        uint64_t j = 0;
        for (uint64_t p = 0; p < n_pages; p++)
            if (dirty[p]) D_out[j++] = (uint32_t)p;
    }

    /* step 4: nothing dirty -> nothing appended, no commit record */
    if (k == 0) { free(dirty); return ORC_OK; }

    /* step 5: all-or-nothing capacity check */
    uint64_t need = ORC_COMMIT_BYTES;
    for (uint64_t p = 0; p < n_pages; p++)
        if (dirty[p]) need += ORC_HDR + page_len(N, P, p);
    if (*W + need > C) { free(dirty); return ORC_ERR_LOG_FULL; }

    /* step 6: page records in ascending page order */
    uint64_t off = *W;
    for (uint64_t p = 0; p < n_pages; p++) {
        if (!dirty[p]) continue;
        uint64_t len = page_len(N, P, p);
        const uint8_t *src = cur + p * P;
        put_u32(log + off + 0, region_id);
        put_u32(log + off + 4, (uint32_t)p);
        put_u32(log + off + 8, (uint32_t)len);
        put_u32(log + off + 12, orc_crc32c(src, len));
        memcpy(log + off + ORC_HDR, src, len);
        off += ORC_HDR + len;
    }

    /* step 7: commit record */
    uint8_t cp[16];
    put_u64(cp + 0, epoch);
    put_u32(cp + 8, region_id);
    put_u32(cp + 12, (uint32_t)k);
    put_u32(log + off + 0, ORC_COMMIT_ID);
    put_u32(log + off + 4, ORC_COMMIT_ID);
    put_u32(log + off + 8, 16u);
    put_u32(log + off + 12, orc_crc32c(cp, 16));
    memcpy(log + off + ORC_HDR, cp, 16);
    off += ORC_COMMIT_BYTES;

    /* step 8: shadow update of the dirty pages */
    for (uint64_t p = 0; p < n_pages; p++)
        if (dirty[p]) memcpy(shadow + p * P, cur + p * P, page_len(N, P, p));

    /* step 9: publish */
    *bytes_out = off - *W;
    *W = off;
    free(dirty);
    return ORC_OK;
}

/* ----------------------------------------------------------------- apply --- */

/* A page record may carry a RUN of consecutive pages ("contiguous dirty ranges use
 * run-length encoding"; reading #38): {region_id, first page, len, crc32c} + len payload
 * bytes, where the payload is the pages first, first+1, ... back to back.  (page_idx, len) is
 * well-formed iff it denotes a whole number (>= 1) of pages inside the region: len > 0, the range
 * [page_idx*P, page_idx*P + len) lies in the region and ends on a page boundary or at the region's
 * end.  A single-page record is the run of length one, so every log of the first format is valid. */
static int rec_len_ok(uint64_t N, uint64_t P, uint64_t pidx, uint64_t len) {
    uint64_t n_pages = (N + P - 1) / P;
    if (pidx >= n_pages || len == 0) return 0;
    uint64_t start = pidx * P;
    if (len > N - start) return 0;
    return (len % P == 0) || (start + len == N);
}

typedef struct {
    uint32_t region_id;
    uint32_t page_bytes;
    uint64_t bytes;
    uint8_t *base;
    uint8_t *shadow; /* may be NULL: then only base is written */
} orc_region;

static const orc_region *find_region(const orc_region *r, uint32_t n, uint32_t id) {
    for (uint32_t i = 0; i < n; i++)
        if (r[i].region_id == id) return &r[i];
    return NULL;
}

/* Apply oracle (SURVEY.md 8c pseudocode).
 * Walks the log record by record; page records are held pending until their
 * commit record validates, then written in log order into base and shadow.
 * A log that runs out of bytes is torn: the committed prefix stays applied and
 * the status is OK.  Any failed check is ORC_ERR_CORRUPT: the committed prefix
 * before the bad epoch stays applied, nothing after it is.
 *   *applied  : page records applied (counting duplicates)
 *   *consumed : offset just after the last applied commit record */
int32_t orc_apply(const uint8_t *log, uint64_t n, const orc_region *regions, uint32_t n_regions,
                  uint64_t *applied, uint64_t *consumed) {
    uint64_t off = 0;
    uint64_t pend_cap = 1024, pend_n = 0;
    uint64_t *pend = (uint64_t *)malloc(pend_cap * sizeof(uint64_t)); /* offsets of pending headers */
    int32_t status = ORC_OK;
    *applied = 0;
    *consumed = 0;
    if (!pend) return ORC_ERR_INVALID;

    for (;;) {
        if (n - off < ORC_HDR) break;                         /* torn */
        const uint8_t *h = log + off;
        uint32_t rid = get_u32(h + 0), pidx = get_u32(h + 4), len = get_u32(h + 8), crc = get_u32(h + 12);
        if ((uint64_t)len > n - off - ORC_HDR) break;         /* torn */
        const uint8_t *payload = h + ORC_HDR;

        if (rid == ORC_COMMIT_ID) {
            int ok = (pidx == ORC_COMMIT_ID) && (len == 16u) && (orc_crc32c(payload, 16) == crc);
            if (ok) {
                uint32_t c_region = get_u32(payload + 8), c_k = get_u32(payload + 12);
                if ((uint64_t)c_k != pend_n) ok = 0;
                for (uint64_t i = 0; ok && i < pend_n; i++)
                    if (get_u32(log + pend[i]) != c_region) ok = 0;
            }
            if (!ok) { status = ORC_ERR_CORRUPT; break; }
            for (uint64_t i = 0; i < pend_n; i++) {
                const uint8_t *ph = log + pend[i];
                const orc_region *r = find_region(regions, n_regions, get_u32(ph + 0));
                uint64_t dst = (uint64_t)get_u32(ph + 4) * r->page_bytes;
                uint32_t plen = get_u32(ph + 8);
                memcpy(r->base + dst, ph + ORC_HDR, plen);
                if (r->shadow) memcpy(r->shadow + dst, ph + ORC_HDR, plen);
            }
            *applied += pend_n;
            off += ORC_COMMIT_BYTES;
            *consumed = off;
            pend_n = 0;
        } else {
            const orc_region *r = find_region(regions, n_regions, rid);
            int ok = (r != NULL);
            if (ok) {
                uint64_t n_pages = (r->bytes + r->page_bytes - 1) / r->page_bytes;
                (void)n_pages;
                ok = rec_len_ok(r->bytes, r->page_bytes, pidx, len) && (orc_crc32c(payload, len) == crc);
            }
            if (!ok) { status = ORC_ERR_CORRUPT; break; }
            if (pend_n == pend_cap) {
                pend_cap *= 2;
                uint64_t *np = (uint64_t *)realloc(pend, pend_cap * sizeof(uint64_t));
                if (!np) { free(pend); return ORC_ERR_INVALID; }
                pend = np;
            }
            pend[pend_n++] = off;
            off += ORC_HDR + len;
        }
    }
    free(pend);
    return status;   /* uncommitted pending records are dropped silently */
}

/* ------------------------------------------------ record writer (config 5a) --- */

/* Append one committed epoch made of caller-given page records: pages[i] is a
 * page index of the region, payloads points at k consecutive payloads of
 * len_p(pages[i]) bytes each.  Same bytes as steps 6-7 above; used by the
 * recovery workload generator ("log written by the oracle's
 * record writer").  No shadow involved. */
int32_t orc_write_epoch(uint8_t *log, uint64_t C, uint64_t *W, uint32_t region_id, uint64_t epoch,
                        uint64_t N, uint64_t P, const uint32_t *pages, uint64_t k, const uint8_t *payloads) {
    uint64_t need = ORC_COMMIT_BYTES;
    for (uint64_t i = 0; i < k; i++) need += ORC_HDR + page_len(N, P, pages[i]);
    if (*W + need > C) return ORC_ERR_LOG_FULL;
    uint64_t off = *W;
    const uint8_t *src = payloads;
    for (uint64_t i = 0; i < k; i++) {
        uint64_t len = page_len(N, P, pages[i]);
        put_u32(log + off + 0, region_id);
        put_u32(log + off + 4, pages[i]);
        put_u32(log + off + 8, (uint32_t)len);
        put_u32(log + off + 12, orc_crc32c(src, len));
        memcpy(log + off + ORC_HDR, src, len);
        off += ORC_HDR + len;
        src += len;
    }
    uint8_t cp[16];
    put_u64(cp + 0, epoch);
    put_u32(cp + 8, region_id);
    put_u32(cp + 12, (uint32_t)k);
    put_u32(log + off + 0, ORC_COMMIT_ID);
    put_u32(log + off + 4, ORC_COMMIT_ID);
    put_u32(log + off + 8, 16u);
    put_u32(log + off + 12, orc_crc32c(cp, 16));
    memcpy(log + off + ORC_HDR, cp, 16);
    *W = off + ORC_COMMIT_BYTES;
    return ORC_OK;
}

/* --------------------------------------- page-range-partitioned scan (mt) --- */

typedef struct {
    const uint8_t *cur, *shadow;
    uint64_t N, P, p0, p1;
    uint8_t *dirty;
    uint64_t k;
} orc_mt_arg;

static void *orc_mt_body(void *v) {
    orc_mt_arg *a = (orc_mt_arg *)v;
    uint64_t k = 0;
    for (uint64_t p = a->p0; p < a->p1; p++) {
        int d = memcmp(a->cur + p * a->P, a->shadow + p * a->P, page_len(a->N, a->P, p)) != 0;
        a->dirty[p] = (uint8_t)d;
        k += (uint64_t)d;
    }
    a->k = k;
    return NULL;
}

/* Same loop as orc_scan with the page range split over n_threads pthreads
 * (BASELINE.md "page-range-partitioned over all cores").  Returns k. */
uint64_t orc_scan_mt(const uint8_t *cur, const uint8_t *shadow, uint64_t N, uint64_t P, uint8_t *dirty,
                     uint32_t n_threads) {
    uint64_t n_pages = (N + P - 1) / P;
    if (n_threads == 0) n_threads = 1;
    if (n_threads > 256) n_threads = 256;
    pthread_t th[256];
    orc_mt_arg arg[256];
    uint64_t per = (n_pages + n_threads - 1) / n_threads;
    for (uint32_t t = 0; t < n_threads; t++) {
        uint64_t p0 = (uint64_t)t * per, p1 = p0 + per;
        if (p0 > n_pages) p0 = n_pages;
        if (p1 > n_pages) p1 = n_pages;
        arg[t] = (orc_mt_arg){cur, shadow, N, P, p0, p1, dirty, 0};
        pthread_create(&th[t], NULL, orc_mt_body, &arg[t]);
    }
    uint64_t k = 0;
    for (uint32_t t = 0; t < n_threads; t++) {
        pthread_join(th[t], NULL);
        k += arg[t].k;
    }
    return k;
}

/* ------------------------- allocator-aware discovery --- */

/* The paper's second discovery policy ("the serving runtime exposes the block
 * table, allocation bitmap, and optional dirty-block/version metadata ... falls back to page
 * diffing only when such metadata is unavailable"; L257 "Allocator-aware regions ... use
 * block-table version counters or dirty-block bitmaps supplied by the serving runtime;
 * Concordia then copies the marked physical pages"; L261 "reads allocator dirty metadata or
 * compares ..."; L264 "Allocator version counters are advanced"; L266 "discovery is
 * proportional to the dirty block bitmap").  Readings (#29-#32):
 *   marked  : packed bitmap, page p = bit (p & 31) of little-endian u32 word p >> 5; bits at
 *             or beyond n_pages are ignored.
 *   verify=0: D = marked pages ("copies the marked physical pages"): a marked page is logged
 *             even when its bytes equal the shadow.
 *   verify=1: D = marked pages whose bytes differ from the shadow (the mark narrows the diff).
 *   shadow  : may be NULL with verify=0 (allocator-aware regions need no shadow); when present
 *             it is refreshed for the pages in D exactly as in orc_checkpoint step 8.
 *   consume : on ORC_OK every word of `marked` is cleared (the runtime's bitmap is handed back
 *             empty); on ORC_ERR_LOG_FULL it is left alone so that a retry sees the same marks.
 * Steps 4-9 (empty epoch, capacity check, records, commit, shadow, publish) are those of
 * orc_checkpoint, written out again rather than shared. */
static int marked_bit(const uint8_t *bm, uint64_t p) {
    uint32_t w = get_u32(bm + 4 * (p >> 5));
    return (int)((w >> (p & 31u)) & 1u);
}

static int32_t append_flagged(const uint8_t *cur, uint8_t *shadow, uint64_t N, uint64_t P, uint32_t region_id,
                              uint64_t epoch, const uint8_t *dirty, uint64_t k, uint8_t *log, uint64_t C,
                              uint64_t *W, uint64_t *bytes_out) {
    uint64_t n_pages = (N + P - 1) / P;
    uint64_t need = ORC_COMMIT_BYTES;
    for (uint64_t p = 0; p < n_pages; p++)
        if (dirty[p]) need += ORC_HDR + page_len(N, P, p);
    if (*W + need > C) return ORC_ERR_LOG_FULL;
    uint64_t off = *W;
    for (uint64_t p = 0; p < n_pages; p++) {
        if (!dirty[p]) continue;
        uint64_t len = page_len(N, P, p);
        const uint8_t *src = cur + p * P;
        put_u32(log + off + 0, region_id);
        put_u32(log + off + 4, (uint32_t)p);
        put_u32(log + off + 8, (uint32_t)len);
        put_u32(log + off + 12, orc_crc32c(src, len));
        memcpy(log + off + ORC_HDR, src, len);
        off += ORC_HDR + len;
    }
    uint8_t cp[16];
    put_u64(cp + 0, epoch);
    put_u32(cp + 8, region_id);
    put_u32(cp + 12, (uint32_t)k);
    put_u32(log + off + 0, ORC_COMMIT_ID);
    put_u32(log + off + 4, ORC_COMMIT_ID);
    put_u32(log + off + 8, 16u);
    put_u32(log + off + 12, orc_crc32c(cp, 16));
    memcpy(log + off + ORC_HDR, cp, 16);
    off += ORC_COMMIT_BYTES;
    if (shadow)
        for (uint64_t p = 0; p < n_pages; p++)
            if (dirty[p]) memcpy(shadow + p * P, cur + p * P, page_len(N, P, p));
    *bytes_out = off - *W;
    *W = off;
    return ORC_OK;
}

int32_t orc_checkpoint_marked(const uint8_t *cur, uint8_t *shadow, uint64_t N, uint64_t P,
                              uint32_t region_id, uint64_t epoch, uint8_t *marked, int verify, int consume,
                              uint8_t *log, uint64_t C, uint64_t *W,
                              uint32_t *D_out, uint64_t *k_out, uint64_t *bytes_out) {
    if (P == 0 || N == 0 || region_id == 0 || region_id == ORC_COMMIT_ID) return ORC_ERR_INVALID;
    if (verify && !shadow) return ORC_ERR_INVALID;
    uint64_t n_pages = (N + P - 1) / P;
    if (n_pages > 0xFFFFFFFEull) return ORC_ERR_INVALID;
    uint8_t *dirty = (uint8_t *)malloc(n_pages);
    if (!dirty) return ORC_ERR_INVALID;
    uint64_t k = 0;
    for (uint64_t p = 0; p < n_pages; p++) {
        int d = marked_bit(marked, p);
        if (d && verify) d = memcmp(cur + p * P, shadow + p * P, page_len(N, P, p)) != 0;
        dirty[p] = (uint8_t)d;
        if (d) { if (D_out) D_out[k] = (uint32_t)p; k++; }
    }
    *k_out = k;
    *bytes_out = 0;
    int32_t st = ORC_OK;
    if (k != 0) st = append_flagged(cur, shadow, N, P, region_id, epoch, dirty, k, log, C, W, bytes_out);
    if (st == ORC_OK && consume) memset(marked, 0, 4 * ((n_pages + 31) / 32));
    free(dirty);
    return st;
}

/* Version-counter form of the same policy (L257 "block-table version counters", L264 "Allocator
 * version counters are advanced"): page p is dirty iff version[p] != committed[p]; after a
 * successful append committed[p] := version[p] for the pages in D (on LOG_FULL nothing moves). */
int32_t orc_checkpoint_versions(const uint8_t *cur, uint8_t *shadow, uint64_t N, uint64_t P,
                                uint32_t region_id, uint64_t epoch, const uint64_t *version, uint64_t *committed,
                                uint8_t *log, uint64_t C, uint64_t *W,
                                uint32_t *D_out, uint64_t *k_out, uint64_t *bytes_out) {
    if (P == 0 || N == 0 || region_id == 0 || region_id == ORC_COMMIT_ID) return ORC_ERR_INVALID;
    uint64_t n_pages = (N + P - 1) / P;
    if (n_pages > 0xFFFFFFFEull) return ORC_ERR_INVALID;
    uint8_t *dirty = (uint8_t *)malloc(n_pages);
    if (!dirty) return ORC_ERR_INVALID;
    uint64_t k = 0;
    for (uint64_t p = 0; p < n_pages; p++) {
        int d = version[p] != committed[p];
        dirty[p] = (uint8_t)d;
        if (d) { if (D_out) D_out[k] = (uint32_t)p; k++; }
    }
    *k_out = k;
    *bytes_out = 0;
    int32_t st = ORC_OK;
    if (k != 0) st = append_flagged(cur, shadow, N, P, region_id, epoch, dirty, k, log, C, W, bytes_out);
    if (st == ORC_OK)
        for (uint64_t p = 0; p < n_pages; p++)
            if (dirty[p]) committed[p] = version[p];
    free(dirty);
    return st;
}

/* ------------------------------ base snapshot + log compactor --- */

/* Base snapshot ("The initial base snapshot captured all 8,192 pages of the full
 * region"; L257 "Immutable regions ... are included in the base snapshot but do not keep GPU
 * shadows"): one committed epoch holding EVERY page of the region, ascending, in the same record
 * format.  If a shadow is given it becomes a copy of the region (the next delta is relative to the
 * snapshot).  Same all-or-nothing capacity rule as orc_checkpoint. */
int32_t orc_snapshot(const uint8_t *cur, uint8_t *shadow, uint64_t N, uint64_t P, uint32_t region_id, uint64_t epoch,
                     uint8_t *log, uint64_t C, uint64_t *W, uint64_t *k_out, uint64_t *bytes_out) {
    if (P == 0 || N == 0 || region_id == 0 || region_id == ORC_COMMIT_ID) return ORC_ERR_INVALID;
    uint64_t n_pages = (N + P - 1) / P;
    if (n_pages > 0xFFFFFFFEull) return ORC_ERR_INVALID;
    uint8_t *all = (uint8_t *)malloc(n_pages);
    if (!all) return ORC_ERR_INVALID;
    memset(all, 1, n_pages);
    *k_out = n_pages;
    *bytes_out = 0;
    int32_t st = append_flagged(cur, shadow, N, P, region_id, epoch, all, n_pages, log, C, W, bytes_out);
    free(all);
    return st;
}

/* Log compactor ("periodic compaction rewrites the log into a smaller base snapshot plus
 * recent deltas"; L87 "a background compactor periodically rewrites the log into a consolidated base
 * snapshot plus a short suffix of deltas"; L221, L266 "bounding replay time").  Readings (DESIGN.md
 * #33-#36): the input is walked and validated exactly as orc_apply walks it (same torn / corrupt
 * rules); within its committed prefix the LAST record of every page survives (what a replay would
 * leave in that page); the output holds, for every region that has a surviving record, in ascending
 * region_id order, ONE committed epoch: one single-page record per surviving page in ascending page
 * order (region_id, page_idx, len, crc32c of the page's bytes; for a page that came from a
 * single-page record this is that record byte for byte, for a page out of a run record it is cut
 * out of the run) and a commit record carrying the epoch
 * number of the last input epoch that touched the region and k = number of surviving pages.
 * A failed check makes the call ORC_ERR_CORRUPT and writes nothing (compaction must not launder a
 * damaged log); a torn tail is dropped (it holds no committed data); ORC_ERR_LOG_FULL writes nothing.
 *   *consumed : bytes of the input covered (end of its last committed epoch)
 *   *n_out    : page records written;  *bytes_out : bytes written at out[0..) */
int32_t orc_compact_log(const uint8_t *log, uint64_t n, const orc_region *regions, uint32_t n_regions,
                        uint8_t *out, uint64_t C_out, uint64_t *bytes_out, uint64_t *consumed, uint64_t *n_out) {
    *bytes_out = 0; *consumed = 0; *n_out = 0;
    if (n_regions == 0 || n_regions > 4096) return ORC_ERR_INVALID;
    uint64_t **last = (uint64_t **)calloc(n_regions, sizeof(uint64_t *));   /* header offset + 1 of the last record, 0 = none */
    uint64_t *last_epoch = (uint64_t *)calloc(n_regions, sizeof(uint64_t));
    uint64_t pend_cap = 1024, pend_n = 0;
    uint64_t *pend = (uint64_t *)malloc(pend_cap * sizeof(uint64_t));
    int32_t status = ORC_OK;
    for (uint32_t i = 0; i < n_regions; i++) {
        uint64_t np = (regions[i].bytes + regions[i].page_bytes - 1) / regions[i].page_bytes;
        last[i] = (uint64_t *)calloc(np, sizeof(uint64_t));
    }
    uint64_t off = 0;
    for (;;) {
        if (n - off < ORC_HDR) break;
        const uint8_t *h = log + off;
        uint32_t rid = get_u32(h + 0), pidx = get_u32(h + 4), len = get_u32(h + 8), crc = get_u32(h + 12);
        if ((uint64_t)len > n - off - ORC_HDR) break;
        const uint8_t *payload = h + ORC_HDR;
        if (rid == ORC_COMMIT_ID) {
            int ok = (pidx == ORC_COMMIT_ID) && (len == 16u) && (orc_crc32c(payload, 16) == crc);
            uint32_t c_region = 0;
            if (ok) {
                c_region = get_u32(payload + 8);
                if ((uint64_t)get_u32(payload + 12) != pend_n) ok = 0;
                for (uint64_t i = 0; ok && i < pend_n; i++)
                    if (get_u32(log + pend[i]) != c_region) ok = 0;
            }
            if (!ok) { status = ORC_ERR_CORRUPT; break; }
            for (uint64_t i = 0; i < pend_n; i++) {
                const uint8_t *ph = log + pend[i];
                uint32_t ri = (uint32_t)(find_region(regions, n_regions, get_u32(ph + 0)) - regions);
                uint64_t P = regions[ri].page_bytes, first = get_u32(ph + 4), rlen = get_u32(ph + 8);
                for (uint64_t q = 0; q * P < rlen; q++)                 /* every page of the run; later records overwrite */
                    last[ri][first + q] = (pend[i] + ORC_HDR + q * P) + 1;     /* offset of the page's payload, + 1 */
                last_epoch[ri] = (uint64_t)get_u32(payload + 0) | ((uint64_t)get_u32(payload + 4) << 32);
            }
            off += ORC_COMMIT_BYTES;
            *consumed = off;
            pend_n = 0;
        } else {
            const orc_region *r = find_region(regions, n_regions, rid);
            int ok = (r != NULL);
            if (ok) {
                uint64_t n_pages = (r->bytes + r->page_bytes - 1) / r->page_bytes;
                (void)n_pages;
                ok = rec_len_ok(r->bytes, r->page_bytes, pidx, len) && (orc_crc32c(payload, len) == crc);
            }
            if (!ok) { status = ORC_ERR_CORRUPT; break; }
            if (pend_n == pend_cap) {
                uint64_t *grown = (uint64_t *)realloc(pend, 2 * pend_cap * sizeof(uint64_t));
                if (!grown) { status = ORC_ERR_INVALID; break; }     /* out of host memory: report, do not crash */
                pend = grown;
                pend_cap *= 2;
            }
            pend[pend_n++] = off;
            off += ORC_HDR + len;
        }
    }
    if (status == ORC_OK) {
        /* size, then all-or-nothing capacity check */
        uint64_t need = 0;
        for (uint32_t i = 0; i < n_regions; i++) {
            uint64_t np = (regions[i].bytes + regions[i].page_bytes - 1) / regions[i].page_bytes, k = 0;
            for (uint64_t p = 0; p < np; p++)
                if (last[i][p]) { need += ORC_HDR + page_len(regions[i].bytes, regions[i].page_bytes, p); k++; }
            if (k) need += ORC_COMMIT_BYTES;
        }
        if (need > C_out) status = ORC_ERR_LOG_FULL;
        else {
            uint64_t o = 0;
            uint32_t prev_id = 0;
            for (;;) {                                   /* regions in ascending region_id order */
                uint32_t best = n_regions;
                for (uint32_t i = 0; i < n_regions; i++)
                    if (regions[i].region_id > prev_id && (best == n_regions || regions[i].region_id < regions[best].region_id))
                        best = i;
                if (best == n_regions) break;
                prev_id = regions[best].region_id;
                uint64_t np = (regions[best].bytes + regions[best].page_bytes - 1) / regions[best].page_bytes, k = 0;
                for (uint64_t p = 0; p < np; p++) {
                    if (!last[best][p]) continue;
                    const uint8_t *pp = log + (last[best][p] - 1);      /* the page's payload inside its record */
                    uint64_t plen = page_len(regions[best].bytes, regions[best].page_bytes, p);
                    put_u32(out + o + 0, regions[best].region_id);
                    put_u32(out + o + 4, (uint32_t)p);
                    put_u32(out + o + 8, (uint32_t)plen);
                    put_u32(out + o + 12, orc_crc32c(pp, plen));
                    memcpy(out + o + ORC_HDR, pp, plen);
                    o += ORC_HDR + plen;
                    k++;
                }
                if (!k) continue;
                uint8_t cp[16];
                put_u64(cp + 0, last_epoch[best]);
                put_u32(cp + 8, regions[best].region_id);
                put_u32(cp + 12, (uint32_t)k);
                put_u32(out + o + 0, ORC_COMMIT_ID);
                put_u32(out + o + 4, ORC_COMMIT_ID);
                put_u32(out + o + 8, 16u);
                put_u32(out + o + 12, orc_crc32c(cp, 16));
                memcpy(out + o + ORC_HDR, cp, 16);
                o += ORC_COMMIT_BYTES;
                *n_out += k;
            }
            *bytes_out = o;
        }
    }
    for (uint32_t i = 0; i < n_regions; i++) free(last[i]);
    free(last); free(last_epoch); free(pend);
    if (status != ORC_OK) *n_out = 0;
    return status;
}

/* ------------------- multi-region checkpoint at one boundary --- */

/* PAPER.md:L259 "At each NCCL or kernel boundary, a four-stage GPU-side pipeline executes" over the
 * registered mutable regions (L217, L257).  Reading (#37): one boundary = one call; the
 * regions that have a shadow are delta-checkpointed one after the other in ascending region_id order,
 * every one exactly as orc_checkpoint does it, all with the same epoch number, each with its own
 * commit record (reading #8: one region per epoch record), the log offset running through.  A region
 * whose records do not fit is skipped whole (its own all-or-nothing rule, shadow untouched); the
 * regions after it are still tried.  Regions without a shadow (allocator-aware, immutable) take no
 * part.  k_out[i] / st_out[i] are per region in the order of `regions`.
 * Returns ORC_OK or the status of the first (lowest id) region that failed. */
int32_t orc_checkpoint_all(const orc_region *regions, uint32_t n_regions, uint64_t epoch,
                           uint8_t *log, uint64_t C, uint64_t *W,
                           uint64_t *k_out, int32_t *st_out, uint64_t *k_total, uint64_t *bytes_total) {
    int32_t first_bad = ORC_OK;
    uint32_t prev_id = 0;
    *k_total = 0;
    *bytes_total = 0;
    for (uint32_t i = 0; i < n_regions; i++) { k_out[i] = 0; st_out[i] = ORC_OK; }
    for (;;) {
        uint32_t best = n_regions;
        for (uint32_t i = 0; i < n_regions; i++)
            if (regions[i].region_id > prev_id && (best == n_regions || regions[i].region_id < regions[best].region_id))
                best = i;
        if (best == n_regions) break;
        prev_id = regions[best].region_id;
        const orc_region *r = &regions[best];
        if (!r->shadow) continue;
        uint64_t k = 0, nb = 0;
        int32_t st = orc_checkpoint(r->base, r->shadow, r->bytes, r->page_bytes, r->region_id, epoch, log, C, W,
                                    NULL, &k, &nb);
        k_out[best] = k;
        st_out[best] = st;
        *k_total += k;
        *bytes_total += nb;
        if (st != ORC_OK && first_bad == ORC_OK) first_bad = st;
    }
    return first_bad;
}

/* --------------------------- run-length records --- */

/* Delta checkpoint with run records ("contiguous dirty ranges use run-length encoding", L221).
 * Same steps as orc_checkpoint except step 6: the ascending dirty pages are grouped into RUNS of
 * consecutive pages; a run never crosses a page index that is a multiple of run_pages (so a run has at
 * most run_pages pages and its byte length fits the u32 len field; run_pages >= 1, run_pages * P <
 * 2^32).  Each run is ONE record {region_id, first page, len = bytes of the whole run,
 * crc32c(all payload bytes of the run)} + the run's pages back to back.  The commit record's count
 * is the number of RECORDS (runs).  run_pages = 1 gives exactly orc_checkpoint's bytes.
 *   *k_out = dirty pages, *runs_out = records written (also on LOG_FULL: what would be written). */
int32_t orc_checkpoint_rle(const uint8_t *cur, uint8_t *shadow, uint64_t N, uint64_t P,
                           uint32_t region_id, uint64_t epoch, uint64_t run_pages,
                           uint8_t *log, uint64_t C, uint64_t *W,
                           uint32_t *D_out, uint64_t *k_out, uint64_t *runs_out, uint64_t *bytes_out) {
    if (P == 0 || N == 0 || region_id == 0 || region_id == ORC_COMMIT_ID) return ORC_ERR_INVALID;
    if (run_pages == 0 || run_pages * P > 0xFFFFFFFFull) return ORC_ERR_INVALID;
    uint64_t n_pages = (N + P - 1) / P;
    if (n_pages > 0xFFFFFFFEull) return ORC_ERR_INVALID;
    uint8_t *dirty = (uint8_t *)malloc(n_pages);
    if (!dirty) return ORC_ERR_INVALID;
    uint64_t k = orc_scan(cur, shadow, N, P, dirty);
    *k_out = k;
    *bytes_out = 0;
    /* a page starts a run iff it is dirty and (it is page 0, or the page before it is clean, or its
     * index is a multiple of run_pages) */
    uint64_t runs = 0, need = ORC_COMMIT_BYTES, j = 0;
    for (uint64_t p = 0; p < n_pages; p++) {
        if (!dirty[p]) continue;
        if (D_out) D_out[j++] = (uint32_t)p;
        if (p == 0 || !dirty[p - 1] || p % run_pages == 0) { runs++; need += ORC_HDR; }
        need += page_len(N, P, p);
    }
    *runs_out = runs;
    if (k == 0) { free(dirty); return ORC_OK; }
    if (*W + need > C) { free(dirty); return ORC_ERR_LOG_FULL; }
    uint64_t off = *W;
    for (uint64_t p = 0; p < n_pages; ) {
        if (!dirty[p]) { p++; continue; }
        uint64_t q = p + 1;                                  /* the run is [p, q) */
        while (q < n_pages && dirty[q] && q % run_pages != 0) q++;
        uint64_t len = (q == n_pages ? N : q * P) - p * P;
        put_u32(log + off + 0, region_id);
        put_u32(log + off + 4, (uint32_t)p);
        put_u32(log + off + 8, (uint32_t)len);
        put_u32(log + off + 12, orc_crc32c(cur + p * P, len));
        memcpy(log + off + ORC_HDR, cur + p * P, len);
        off += ORC_HDR + len;
        p = q;
    }
    uint8_t cp[16];
    put_u64(cp + 0, epoch);
    put_u32(cp + 8, region_id);
    put_u32(cp + 12, (uint32_t)runs);
    put_u32(log + off + 0, ORC_COMMIT_ID);
    put_u32(log + off + 4, ORC_COMMIT_ID);
    put_u32(log + off + 8, 16u);
    put_u32(log + off + 12, orc_crc32c(cp, 16));
    memcpy(log + off + ORC_HDR, cp, 16);
    off += ORC_COMMIT_BYTES;
    for (uint64_t p = 0; p < n_pages; p++)
        if (dirty[p]) memcpy(shadow + p * P, cur + p * P, page_len(N, P, p));
    *bytes_out = off - *W;
    *W = off;
    free(dirty);
    return ORC_OK;
}
