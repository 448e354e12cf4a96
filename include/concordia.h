/*
 * concordia.h -- C ABI of libconcordia.so: GPU-side delta checkpointing of registered
 * regions on one NVIDIA B200 (sm_100a).
 *
 * The operations are those of Concordia (arxiv 2606.23521; citations are lines of
 * /root/reference/PAPER.md as used in SURVEY.md / DESIGN.md):
 *   - region registration              PAPER.md:L193 (region specification), L217 (registered regions)
 *   - delta checkpoint                 PAPER.md:L219, L259-264 (4-stage pipeline: dirty discovery ->
 *                                      record construction -> append + commit -> shadow update)
 *   - append-only log discipline       PAPER.md:L221 (header, payloads, commit marker, publish epoch;
 *                                      recovery ignores an uncommitted suffix)
 *   - recovery applier                 PAPER.md:L156-158 (TASK_RESTORE), L227, L445
 *   - ring buffer + persistent worker  PAPER.md:L119, L125-160 (listings), L247-249 (host-mapped
 *                                      memory, release/acquire), Table 1 L166-175 (host API)
 *   - allocator-aware discovery        PAPER.md:L217, L257, L261, L264, L266 (dirty bitmaps / version counters)
 *   - run-length records               PAPER.md:L221 ("contiguous dirty ranges use run-length encoding")
 *   - base snapshot + log compactor
 *   - all regions at one boundary      PAPER.md:L259 ("at each NCCL or kernel boundary")
 *   - staging buffer -> host log       PAPER.md:L262-263 (cc_log_mirror_attach / cc_log_drain)
 *
 * Conventions
 *   - Plain C, no exceptions across the boundary.  Every call returns an int32_t status:
 *     CC_OK (0) or a negative CC_ERR_*; on error there are no partial side effects unless
 *     stated.  cc_poll returns CC_PENDING (1) while a task is still running.
 *   - OWNERSHIP: the caller owns, and keeps alive, every buffer it passes (live region,
 *     shadow, workspace, log buffer, apply scratch, result structs).  The library borrows the
 *     pointers.  It allocates its own small control blocks in cc_init / cc_worker_start only
 *     and never allocates or frees device memory while the worker is running
 *     (cudaMalloc / cudaDeviceSynchronize can deadlock under a resident kernel).
 *   - "device" pointers are CUDA device memory of the context's GPU.  "pinned host" pointers
 *     are page-locked, device-mapped host memory (cudaHostAlloc / torch pin_memory; with UVA
 *     the same address is valid on both sides).  A log buffer and a cc_result
 *     may be either; regions, shadows, workspaces and apply scratch are device memory.
 *   - Streams are cudaStream_t passed as void* (0 = the legacy default stream).
 *   - One host thread per context at a time (cc_submit is single-producer).
 *   - No CPU fallback exists: if no CUDA device is usable cc_init fails with CC_ERR_CUDA.
 *
 * On-log record format (the paper lists the fields, PAPER.md:L85,
 * L219, not their widths).  All integers little-endian, no padding:
 *   page record   : { u32 region_id; u32 page_idx; u32 len; u32 crc32c(payload) } + len payload bytes
 *                   (len = one page, or a run of consecutive pages starting at page_idx: cc_checkpoint_delta_rle)
 *   commit record : { 0xFFFFFFFF; 0xFFFFFFFF; 16; crc32c(payload) } + { u64 epoch; u32 region_id; u32 k }
 *   CRC32C        : Castagnoli, reflected 0x82F63B78, init 0xFFFFFFFF, xorout 0xFFFFFFFF.
 * One checkpoint of one region appends its k dirty pages in ascending page order followed by
 * one commit record, or nothing at all when k == 0.
 */
#ifndef CONCORDIA_H
#define CONCORDIA_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CC_OK 0
#define CC_PENDING 1
#define CC_ERR_INVALID (-1)        /* bad argument / alignment / size */
#define CC_ERR_NOT_REGISTERED (-2)
#define CC_ERR_EXISTS (-3)
#define CC_ERR_LOG_FULL (-4)       /* checkpoint: W + need > capacity; nothing appended, shadow untouched */
#define CC_ERR_CORRUPT (-5)        /* apply: a structure or CRC check failed; committed prefix before it applied */
#define CC_ERR_RING_FULL (-6)
#define CC_ERR_WORKER (-7)         /* worker not running / running when it must not be / heartbeat stale */
#define CC_ERR_CUDA (-8)           /* a CUDA call failed: cc_last_cuda_error() */
#define CC_ERR_TIMEOUT (-9)
#define CC_ERR_SCRATCH (-10)       /* apply: log holds more records/epochs than the attached scratch; nothing applied */
#define CC_ERR_STATIC_LIMIT (-11)  /* cc_dirty_pages_static: the region has more than CC_STATIC_MAX_PAGES pages */

#define CC_MAX_REGIONS 64
#define CC_COMMIT_ID 0xFFFFFFFFu
#define CC_RECORD_HEADER_BYTES 16u
#define CC_COMMIT_RECORD_BYTES 32u

/* cc_region_desc.flags */
#define CC_REG_SNAPSHOT_NOW 1u     /* shadow := base at registration (first delta is relative to now) */
#define CC_REG_NO_SHADOW 2u        /* allocator-aware region: `shadow` is NULL, dirty pages come from
                                      cc_checkpoint_marked / cc_checkpoint_versions only; calls that need the shadow
                                      (cc_checkpoint_delta, cc_scan_only, CC_MARK_VERIFY) return CC_ERR_INVALID */

/* cc_checkpoint_marked flags */
#define CC_MARK_VERIFY 1u          /* compare the marked pages with the shadow and log only those that differ */
#define CC_MARK_CONSUME 2u         /* clear the caller's bitmap once the checkpoint went through (not on LOG_FULL) */

#define CC_WORKER_BLOCKS_DEFAULT 16u /* ~11 % of B200's 148 SMs; the trade-off is tabulated in DESIGN.md section 9 */
#define CC_WORKER_BLOCKS_ALL 0xFFFFFFFFu

typedef struct cc_ctx cc_ctx;

typedef struct {
    uint32_t ring_capacity;    /* slots, power of two, 0 = 256 (256 x 64 B) */
    uint32_t worker_blocks;    /* persistent worker CTAs: 0 = CC_WORKER_BLOCKS_DEFAULT, CC_WORKER_BLOCKS_ALL = as many as are
                                  co-resident with worker_threads (maximum checkpoint bandwidth, every SM taken) */
    uint32_t worker_threads;   /* threads per worker CTA ("tpb" of Table 1), multiple of 32, 0 = 512 */
    uint32_t backoff_ns;       /* idle poll back-off of the worker (set_yield_every analogue, L172), 0 = 500 */
    uint64_t max_lifetime_ns;  /* worker exits by itself after this long (safety net), 0 = 600 s */
} cc_config;

typedef struct {
    uint32_t region_id;        /* 1 ... 0xFFFFFFFE */
    uint32_t page_bytes;       /* P: multiple of 16 (benchmarks: 4096 / 16384 / 65536) */
    uint64_t bytes;            /* N: multiple of 16, > 0; the last page may be short; ceil(N/P) <= 2^31 */
    void*    base;             /* live region, device, 16-byte aligned */
    void*    shadow;           /* last-committed copy, device, N bytes, 16-byte aligned, caller-allocated
                                  (NULL with CC_REG_NO_SHADOW) */
    void*    workspace;        /* device, 256-byte aligned, >= cc_workspace_bytes(N, P); zeroed by the call */
    uint64_t workspace_bytes;
    uint32_t flags;            /* CC_REG_* */
    uint32_t reserved;
} cc_region_desc;

/* Completion / result record, exactly 64 bytes.  Written by the GPU. */
typedef struct {
    uint64_t seq_done;         /* worker path: task seq + 1; host-launched path: 1.  Stored LAST, at system scope, behind a
                                  system-scope fence that covers every other field and every log byte of the call */
    uint64_t n_dirty;          /* checkpoint: k;  apply: page records applied (duplicates counted) */
    uint64_t bytes;            /* checkpoint: bytes appended;  apply: bytes consumed (end of last applied commit) */
    uint64_t log_offset_after; /* checkpoint: log write offset W after the call;  apply: same as bytes */
    uint64_t epoch;            /* checkpoint: the epoch passed in;  apply: number of epochs applied */
    int32_t  status;           /* CC_OK / CC_ERR_LOG_FULL / CC_ERR_CORRUPT / CC_ERR_SCRATCH / ... */
    uint32_t flags;            /* task kind echoed back */
    uint64_t t_start_ns;       /* %globaltimer when the GPU started the operation */
    uint64_t t_end_ns;         /* %globaltimer when it finished */
} cc_result;

/* Task descriptor, exactly 64 bytes ("64-128 bytes including operator ID, tensor
 * pointers, dimensions, and control flags"; L148-159 kinds, epoch, seq). */
#define CC_TASK_NOP 0u
#define CC_TASK_DELTA_CKPT 1u      /* region_id, epoch */
#define CC_TASK_RESTORE 2u         /* arg0 = log pointer, arg1 = nbytes */
#define CC_TASK_LOG_RESET 3u       /* W := 0 */
/* kind 4 is CC_TASK_TEST_MUTATE, a bench / test hook (end of this header) */
#define CC_TASK_MARKED_CKPT 5u     /* region_id, epoch; arg0 = dirty bitmap (device), arg1 = CC_MARK_* flags */
#define CC_TASK_VERSION_CKPT 6u    /* region_id, epoch; arg0 = version[] (device), arg1 = committed[] (device) */
#define CC_TASK_SNAPSHOT 7u        /* region_id, epoch: base snapshot (cc_snapshot_region) */
#define CC_TASK_COMPACT_LOG 8u     /* arg0 = input log, arg1 = its bytes, arg2 = output log, arg3 = output capacity */
#define CC_TASK_CKPT_ALL 9u        /* epoch: every region that has a shadow (cc_checkpoint_all) */
#define CC_TASK_EXIT 255u
#define CC_TASKF_RLE 2u            /* cc_task.flags, CC_TASK_DELTA_CKPT only: run records, arg0 = run_pages (cc_checkpoint_delta_rle) */
#define CC_TASKF_FUSED 1u          /* cc_task.flags, CC_TASK_DELTA_CKPT only: run the fused single pass (cc_checkpoint_delta_fused) */
typedef struct {
    uint32_t kind;
    uint32_t region_id;
    uint32_t flags;
    uint32_t version;          /* carried, unused (the paper's operator-table version) */
    uint64_t seq;              /* assigned by cc_submit */
    uint64_t epoch;
    uint64_t arg0, arg1, arg2, arg3;
} cc_task;

/* ---- lifecycle (Table 1: init / shutdown) --------------------------------------- */

/* Create a context on CUDA device `device`.  cfg may be NULL (all defaults). */
int32_t cc_init(cc_ctx** out, int32_t device, const cc_config* cfg);
/* Stop the worker if it runs, free the library's control blocks.  Caller buffers are untouched. */
int32_t cc_shutdown(cc_ctx* ctx);
/* Last cudaError_t seen by this context (0 = none). */
int32_t cc_last_cuda_error(cc_ctx* ctx);
/* Number of kernels this context has launched so far (host-launched path + worker launches). */
uint64_t cc_kernel_launches(cc_ctx* ctx);

/* ---- regions ------------------------------------------------------- */

/* Device workspace a region of N bytes with pages of P bytes needs (0 if the pair is invalid). */
uint64_t cc_workspace_bytes(uint64_t bytes, uint32_t page_bytes);
/* Register a region.  Synchronous (zeroes the workspace, optionally snapshots the shadow, on an
 * internal stream, and waits).  Only while the worker is stopped (CC_ERR_WORKER otherwise). */
int32_t cc_register_region(cc_ctx* ctx, const cc_region_desc* desc);
int32_t cc_unregister_region(cc_ctx* ctx, uint32_t region_id);

/* ---- log placement ("AOF log placement") ------------------------------------ */

/* Attach the append-only log: log_buf (device or pinned host, 16-byte aligned), capacity bytes.
 * committed_off (pinned host or device, 8 bytes, may be NULL) receives the committed write
 * offset after every commit record: a system-scope store behind ONE system-scope fence that, by cumulativity, covers
 * every record byte the call wrote, whichever block wrote it ("a commit marker publishes the epoch
 * only after all bytes are visible").  A host thread that reads the word with acquire semantics may read the log up to
 * that offset without synchronising with the stream.  W := 0.
 * Only while the worker is stopped. */
int32_t cc_log_attach(cc_ctx* ctx, void* log_buf, uint64_t capacity, uint64_t* committed_off);
/* W := 0 and *committed_off := 0 (synchronous; only while the worker is stopped -- use CC_TASK_LOG_RESET otherwise). */
int32_t cc_log_reset(cc_ctx* ctx);

/* W := 0 and *committed_off := 0, ASYNCHRONOUS on `stream` (ordered after the checkpoints already queued there): what a log
 * drainer calls once it has consumed the committed prefix.  Only while the worker is stopped. */
int32_t cc_log_reset_async(cc_ctx* ctx, void* stream);

/* Host mirror of a DEVICE-resident log, filled by the copy engine (records are built in a
 * staging buffer, then "copied to a CXL-backed or DRAM-backed append-only log; a commit marker publishes the epoch
 * only after all bytes are visible").  With the log attached in device memory a checkpoint appends at HBM speed;
 * cc_log_drain then copies the newly committed bytes [drained, upto) to the same offsets of `host_log` (pinned host
 * memory, 16-byte aligned) with cudaMemcpyAsync on `copy_stream` -- ordered after the work already queued on
 * `after_stream` -- and, once the bytes have landed, release-stores `upto` into *committed_off_host (may be NULL)
 * from a host callback on that stream.  The copy engine reaches the full link rate and takes no SM; the drain
 * of one checkpoint overlaps the scan of the next.  `upto` must be a committed offset the caller has read from a
 * result (cc_result.log_offset_after), non-decreasing between resets.  cc_log_reset rewinds the drain position too;
 * the caller makes sure the copy stream has drained before it resets or reuses log space.  host_log = NULL detaches.
 * CC_ERR_LOG_FULL if upto exceeds the mirror's capacity. */
int32_t cc_log_mirror_attach(cc_ctx* ctx, void* host_log, uint64_t capacity, uint64_t* committed_off_host);
int32_t cc_log_drain(cc_ctx* ctx, uint64_t upto, void* after_stream, void* copy_stream);

/* Library-side drainer for the same mirror: cc_log_drain_start launches a host thread that follows the committed
 * offset every checkpoint publishes (host-launched calls and worker tasks alike -- no per-step call, no result to
 * read first) and hands each newly committed byte range to the copy engine on an internal stream; once a range
 * has landed in host_log, *committed_off_host is release-stored.  A log reset (cc_log_reset, cc_log_reset_async,
 * CC_TASK_LOG_RESET) starts a new generation: the thread starts again at offset 0 and zeroes *committed_off_host.
 * As with cc_log_drain, the caller resets or reuses log space only after the mirror has caught up
 * (cc_log_drain_wait, or poll *committed_off_host).  cc_log_drain_wait blocks until the first `upto` bytes of the
 * current generation have landed (CC_ERR_TIMEOUT after timeout_ns; the thread's error if it stopped:
 * CC_ERR_LOG_FULL = mirror too small, CC_ERR_CUDA).  cc_log_drain_stop drains what is committed, joins the thread
 * and returns its status.  cc_log_drain, cc_log_attach and cc_log_mirror_attach are refused (CC_ERR_INVALID)
 * while the thread runs; cc_shutdown stops it.  Needs an attached log and mirror. */
int32_t cc_log_drain_start(cc_ctx* ctx);
int32_t cc_log_drain_wait(cc_ctx* ctx, uint64_t upto, uint64_t timeout_ns);
int32_t cc_log_drain_stop(cc_ctx* ctx);

/* ---- host-launched path -------------------------------------------------------------------- */

/* One checkpoint of one region -- the general entry point; the named calls below are this call with fixed options.
 *   discovery   where the dirty set comes from: CC_DISC_SCAN compare live vs shadow; CC_DISC_MARKS the
 *               runtime's dirty-page bitmap (L257; mark_flags = CC_MARK_VERIFY / CC_MARK_CONSUME); CC_DISC_VERSIONS
 *               per-page version counters (L257, L264); CC_DISC_ALL every page (base snapshot, L394)
 *   run_pages   0 / 1: one record per dirty page; >= 2: run-length records (L221), a run never crossing a page index
 *               that is a multiple of run_pages (run_pages * page_bytes < 2^32)
 *   path        CC_PATH_SINGLE_PASS: ONE kernel launch -- warp tiles of pages are discovered, ranked by decoupled
 *               look-back and written (records, CRC32C, shadow) by the same warp, the last warp of the grid commits
 *               and publishes; needs run_pages <= 32 and at most 2^20 * (32 rounded down to a multiple of run_pages) pages -- 2^25 for
 *               page records (CC_ERR_INVALID otherwise).  When the
 *               worst case (every page dirty) does not fit behind the log's write offset, the same launch runs the
 *               classic phases behind grid barriers instead (all-or-nothing needs the count first).
 *               CC_PATH_PHASES: the classic phases as separate launches (discovery, ordered compaction,
 *               [run ranking,] gather + commit), each sized for its own work.  For page records on a region of at most
 *               131,072 pages and 1 GiB it is two launches: the scan, then one kernel in which every block ranks the
 *               dirty bitmap by itself and writes its share of the records (no compaction launch).
 *               CC_PATH_SMALL: ONE kernel launch with one grid-wide rendezvous, for regions of at most 131,072 pages
 *               (CC_DISC_SCAN, one record per page; CC_ERR_INVALID otherwise): scan, then every block ranks the
 *               whole dirty bitmap by itself and the record writer follows at once.  It is what the persistent worker
 *               runs for a plain CC_TASK_DELTA_CKPT on such a region; host-launched the two-launch phases are faster.
 *               CC_PATH_AUTO: the phases, except with a pinned host log on regions of 128 MiB and more, where the single
 *               pass sends the records over the host link while it scans.
 * Every path writes the same bytes.  Result, asynchrony, CC_ERR_LOG_FULL rule: as cc_checkpoint_delta below. */
#define CC_DISC_SCAN 0u
#define CC_DISC_MARKS 1u
#define CC_DISC_VERSIONS 3u
#define CC_DISC_ALL 4u
#define CC_PATH_AUTO 0u
#define CC_PATH_SINGLE_PASS 1u
#define CC_PATH_PHASES 2u
#define CC_PATH_SMALL 3u
typedef struct {
    uint32_t discovery;        /* CC_DISC_* */
    uint32_t path;             /* CC_PATH_* */
    uint32_t run_pages;
    uint32_t mark_flags;       /* CC_DISC_MARKS: CC_MARK_* */
    uint32_t* dirty_bitmap;    /* CC_DISC_MARKS: device, ceil(n_pages/32) u32 words */
    const uint64_t* version;   /* CC_DISC_VERSIONS: device, n_pages u64 */
    uint64_t* committed;       /* CC_DISC_VERSIONS: device, n_pages u64, advanced by the call */
} cc_ckpt_opts;
int32_t cc_checkpoint_ex(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, const cc_ckpt_opts* opts /* NULL = all zero */,
                         void* stream, cc_result* out);

/* Delta-checkpoint one region: scan live vs shadow per page, compact the
 * dirty page indices in ascending order, append k page records + one commit record at the log
 * write offset, refresh the shadow of the dirty pages, publish the committed offset.
 * ASYNCHRONOUS on `stream`: kernels only, no host round trip between them.  `out` (pinned host
 * or device, 64 bytes, may be NULL) is valid once the stream has reached this point.
 * k == 0 appends nothing.  If the records do not fit: out->status = CC_ERR_LOG_FULL, nothing is
 * appended and the shadow is untouched.  The return value covers argument / launch errors only.
 * The region must not be written while the call is in flight (boundaries are
 * quiescent).  The ascending dirty list of the last checkpoint stays readable in the workspace
 * (cc_dirty_list). */
int32_t cc_checkpoint_delta(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, void* stream, cc_result* out);

/* Same contract, same log bytes, same result as cc_checkpoint_delta, always by the single pass
 * (cc_checkpoint_ex with CC_PATH_SINGLE_PASS; cc_checkpoint_delta itself is CC_PATH_AUTO). */
int32_t cc_checkpoint_delta_fused(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, void* stream, cc_result* out);

/* Delta checkpoint with RUN-LENGTH records ("Sparse page maps use index-value records;
 * contiguous dirty ranges use run-length encoding"): as cc_checkpoint_delta, but consecutive dirty pages
 * form ONE record { region_id, first page, len = bytes of the whole run, crc32c(all payload bytes of the
 * run) } + the run's pages back to back.  A run never crosses a page index that is a multiple of
 * run_pages (>= 1, run_pages * page_bytes < 2^32), so it has at most run_pages pages; run_pages = 1 gives
 * cc_checkpoint_delta's bytes.  run_pages <= 32 follows CC_PATH_AUTO (single pass where that applies: runs are cut
 * inside a warp tile, whose dirty mask is one register); larger run_pages take the phases.  The commit record counts RECORDS; out->n_dirty still counts pages.
 * cc_apply_log and cc_compact_log read both kinds of record (a single-page record is the run of length
 * one). */
int32_t cc_checkpoint_delta_rle(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, uint32_t run_pages, void* stream,
                                cc_result* out);

/* Allocator-aware delta checkpoint ("reads allocator dirty metadata", L266
 * "discovery is proportional to the dirty block bitmap"): the dirty set comes from the runtime's
 * dirty-page bitmap instead of a scan of the whole region.  `dirty_bitmap` is device memory, 4-byte
 * aligned, ceil(n_pages/32) u32 words; page p is bit (p & 31) of word p >> 5; bits at or beyond
 * n_pages are ignored.  flags = 0: every marked page is logged ("copies the marked physical pages"),
 * whether or not its bytes changed.  CC_MARK_VERIFY: only the marked pages are compared with the
 * shadow and those that differ are logged -- the same log as cc_checkpoint_delta whenever the marks
 * cover the dirty set.  CC_MARK_CONSUME: the bitmap words are zeroed once the checkpoint went through
 * (status CC_OK, an empty epoch included); on CC_ERR_LOG_FULL they are left alone.  Everything else
 * (records, commit, shadow refresh of the logged pages when the region has a shadow, result,
 * asynchrony) is as in cc_checkpoint_delta. */
int32_t cc_checkpoint_marked(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, uint32_t* dirty_bitmap,
                             uint32_t flags, void* stream, cc_result* out);

/* Same, from per-page version counters ("block-table version counters", L264 "Allocator
 * version counters are advanced"): page p is dirty iff version[p] != committed[p] (both device, u64,
 * n_pages entries, 8-byte aligned; `committed` is caller-owned state that only this call writes).
 * After a successful append committed[p] := version[p] for the logged pages; on CC_ERR_LOG_FULL
 * nothing moves. */
int32_t cc_checkpoint_versions(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, const uint64_t* version,
                               uint64_t* committed, void* stream, cc_result* out);

/* One boundary, all regions ("At each NCCL or kernel boundary, a four-stage GPU-side
 * pipeline executes"; L217, L257): every registered region that has a shadow is delta-checkpointed with
 * the same epoch number.  The log receives the regions' epochs in ascending region_id order, each with
 * its own commit record -- the same bytes as calling cc_checkpoint_delta region by region in that order --
 * in four kernel launches whatever the number of regions.  A region whose records do not fit is skipped
 * whole (shadow untouched); the regions after it are still tried.  The committed offset is published once,
 * after every region's commit record is visible.  Result: n_dirty / bytes summed over the regions,
 * log_offset_after = final write offset, status = CC_OK or the status of the lowest-id region that
 * failed; per-region dirty lists through cc_dirty_list.  Regions registered with CC_REG_NO_SHADOW take
 * no part.  ASYNCHRONOUS on `stream`. */
int32_t cc_checkpoint_all(cc_ctx* ctx, uint64_t epoch, void* stream, cc_result* out);

/* The same boundary with RUN-LENGTH records (reading #38): the bytes of calling
 * cc_checkpoint_delta_rle(region, epoch, run_pages) region by region in ascending region_id order.  One launch per
 * region (the single pass for run_pages <= 32, the phases above that) plus one that sums up the result; the committed
 * offset moves region by region, always to the end of a whole epoch.  Skipping rule, result and the regions that
 * take part: as cc_checkpoint_all.  run_pages >= 1 and run_pages * page_bytes < 2^32 for every region taking part
 * (CC_ERR_INVALID otherwise, nothing launched). */
int32_t cc_checkpoint_all_rle(cc_ctx* ctx, uint64_t epoch, uint32_t run_pages, void* stream, cc_result* out);

/* Base snapshot ("The initial base snapshot captured all 8,192 pages of the full region";
 * L257: immutable regions "are included in the base snapshot but do not keep GPU shadows"): append EVERY
 * page of the region, ascending, as one committed epoch in the same record format -- no discovery pass.
 * A region with a shadow gets shadow := base (the next delta is relative to the snapshot).  Same
 * all-or-nothing CC_ERR_LOG_FULL rule, result and asynchrony as cc_checkpoint_delta. */
int32_t cc_snapshot_region(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, void* stream, cc_result* out);

/* Log compactor ("a background compactor periodically rewrites the log into a
 * consolidated base snapshot plus a short suffix of deltas", L221, L266 "bounding replay time").
 * in_log[0, in_bytes) is parsed and validated exactly as cc_apply_log does (same torn / corrupt rules;
 * needs the scratch of cc_apply_attach).  Within its committed prefix the LAST record of every page
 * survives; out_log (device or pinned host, 16-byte aligned, must not overlap in_log) receives, for
 * every region with a surviving record, in ascending region_id order, ONE committed epoch: the
 * surviving page records in ascending page order and a commit record carrying the epoch number of
 * the last input epoch that touched the region.  Replaying out_log leaves every registered region in
 * the state that replaying in_log leaves it in.  Regions and the attached log are not touched.
 * Result: status CC_OK, n_dirty = page records written, bytes = bytes written at out_log[0..),
 * log_offset_after = input bytes covered (end of its last committed epoch), epoch = regions written.
 * CC_ERR_CORRUPT (a failed check anywhere in the input), CC_ERR_SCRATCH and CC_ERR_LOG_FULL
 * (out_capacity too small) write nothing.  ASYNCHRONOUS on `stream`.  The per-region dirty lists
 * (cc_dirty_list) are overwritten. */
int32_t cc_compact_log(cc_ctx* ctx, const void* in_log, uint64_t in_bytes, void* out_log, uint64_t out_capacity,
                       void* stream, cc_result* out);

/* Scan + compaction only (steps a1-a2), for measurement: fills the dirty list, appends nothing,
 * leaves the shadow alone.  out->n_dirty = k. */
int32_t cc_scan_only(cc_ctx* ctx, uint32_t region_id, void* stream, cc_result* out);

/* Device pointer to the u32 ascending dirty page list of the region's last scan and to its
 * u32 count (valid after the stream reached the end of that call). */
int32_t cc_dirty_list(cc_ctx* ctx, uint32_t region_id, const uint32_t** d_list, const uint32_t** d_count);

/* Attach device scratch for the applier: room for the record / epoch tables of a log with at most
 * max_records page records and max_records commit records; cc_apply_scratch_bytes gives the size.
 * Only while the worker is stopped. */
uint64_t cc_apply_scratch_bytes(uint64_t max_records);
int32_t cc_apply_attach(cc_ctx* ctx, void* scratch, uint64_t scratch_bytes);

/* Optional device staging buffer for HOST-resident logs (16-byte aligned device memory; NULL / 0 detaches).
 * The applier and the compactor read a log twice (validate, then scatter / copy).  When the log passed to
 * cc_apply_log / cc_compact_log is pinned host memory of at most `bytes` bytes, it is first copied into this
 * buffer by the copy engine on the call's stream (one pass over the host link at DMA speed) and the kernels
 * read the device copy; results are identical.  Logs that do not fit, device-resident logs and the worker's
 * RESTORE / COMPACT_LOG tasks are unaffected.  Only while the worker is stopped. */
int32_t cc_apply_stage_attach(cc_ctx* ctx, void* device_buf, uint64_t bytes);
/* How often the staging buffer was used since cc_init: *staged = host-resident logs that were copied into it,
 * *bypassed = host-resident logs that were read in place ALTHOUGH a buffer is attached, because they are larger than it
 * or the copy could not be queued.  A bypassed replay is correct but crosses the host link three times instead of once
 * (C5a: 16.9 ms instead of 5.5 ms) -- a caller that sees the second counter move should attach a larger buffer.
 * Either pointer may be NULL. */
int32_t cc_apply_stage_stats(cc_ctx* ctx, uint64_t* staged, uint64_t* bypassed);

/* Recovery applier: parse log[0, nbytes) (device or pinned host,
 * 16-byte aligned), validate structure and CRC32C of every record, and for every committed epoch
 * before the first failed check, in log order, write each page record's payload into its
 * region's live page and shadow page (a page present several times ends with its last record).
 * Running out of bytes is "torn": status CC_OK, the committed prefix is applied.  A failed check
 * is CC_ERR_CORRUPT: the committed prefix before the bad epoch is applied, nothing after.
 * ASYNCHRONOUS on `stream`; result fields as documented in cc_result. */
int32_t cc_apply_log(cc_ctx* ctx, const void* log, uint64_t nbytes, void* stream, cc_result* out);

/* ---- ring buffer + persistent worker ------------------- */

/* Launch the persistent worker kernel (cooperative, stays resident) on an internal non-blocking
 * stream.  Everything (regions, log, apply scratch) must be registered/attached before. */
int32_t cc_worker_start(cc_ctx* ctx);
/* Submit CC_TASK_EXIT, wait for the kernel to leave (up to 10 s), CC_ERR_TIMEOUT otherwise. */
int32_t cc_worker_stop(cc_ctx* ctx);
/* Table 1 worker_alive(): 1 if the worker runs and its heartbeat advanced within 1 s, else 0. */
int32_t cc_worker_alive(cc_ctx* ctx);
/* Footprint of the persistent worker (Table 9): CTAs, threads per CTA, shared memory per CTA, registers
 * per thread, SMs of the device.  Any output pointer may be NULL. */
int32_t cc_worker_footprint(cc_ctx* ctx, uint32_t* blocks, uint32_t* threads, uint32_t* smem_bytes, uint32_t* regs,
                            uint32_t* sm_count);
/* Table 1 peek_queue(): head = tasks completed, tail = tasks submitted. */
int32_t cc_peek_queue(cc_ctx* ctx, uint64_t* head, uint64_t* tail);
/* Copy *task into the next ring slot and publish it with a store-release;
 * no CUDA call.  Non-blocking: CC_ERR_RING_FULL when `capacity` tasks are outstanding.
 * *seq_out (may be NULL) = the sequence number to poll / wait on. */
int32_t cc_submit(cc_ctx* ctx, const cc_task* task, uint64_t* seq_out);
/* CC_OK and *out filled when task `seq` has completed; CC_PENDING otherwise.  A completion slot
 * is reused `capacity` submissions later: poll before then. */
int32_t cc_poll(cc_ctx* ctx, uint64_t seq, cc_result* out);
/* Spin (host) until done or timeout_ns elapsed (CC_ERR_TIMEOUT). */
int32_t cc_wait(cc_ctx* ctx, uint64_t seq, uint64_t timeout_ns, cc_result* out);

/* ---- dirty list without any allocation ---------------------------------------------------- */

/* Steps a1-a2 for callers that cannot allocate: compare `cur` with `shadow` page by page
 * and write the ascending list of the pages that differ -- the list cc_scan_only + cc_dirty_list give -- with
 * NO context, NO registered region, NO workspace, and no cudaMalloc / cudaFree / allocating library routine
 * anywhere in the call.  It is meant for code that runs beside a resident persistent kernel (device allocation
 * synchronises the GPU and can wait forever on a kernel that never exits), for servers whose
 * memory pool took all of HBM at start-up (a later cudaMalloc just fails), and for fault handlers that want to
 * see what changed before they touch any allocator.
 *
 * The scratch (one bit per page + a counter) is a fixed array inside the library image, 2 MiB + 256 bytes,
 * enough for CC_STATIC_MAX_PAGES pages: every GPU that loads libconcordia.so holds it until the process exits.
 * A region with more pages is refused with CC_ERR_STATIC_LIMIT and nothing is launched; use a larger page
 * size, call per sub-range, or use the workspace path.
 *
 *   device         CUDA device ordinal (0 ... 63) that owns every pointer and the stream; made current for the
 *                  duration of the call and the previous device restored
 *   cur, shadow    device memory, `bytes` bytes each, 16-byte aligned; only read
 *   bytes          multiple of 16, > 0;   page_bytes  multiple of 16, > 0;  the last page may be short
 *   d_list         device, u32[list_capacity], caller-owned: receives min(k, list_capacity) ascending page indices
 *                  (may be NULL when list_capacity is 0: count only)
 *   d_count        device (or pinned host), one u32, caller-owned: receives k, the number of dirty pages, even
 *                  when k > list_capacity -- that is how a too-short list shows
 *   stream         cudaStream_t of `device` (0 = legacy default stream).  ASYNCHRONOUS: one memset of the scratch
 *                  and one kernel are queued; outputs are valid once the stream has reached that point
 *   cuda_error     may be NULL; receives the cudaError_t when the return value is CC_ERR_CUDA
 *
 * FIRST CALL ON A DEVICE does the set-up: it resolves the array's device address (cudaGetSymbolAddress) and the
 * launch geometry, which can make the runtime load the library's GPU code.  Make that first call outside any
 * stream capture and before anything that must not stall; later calls only queue work.
 * ONE ARRAY, SHARED: all calls on a GPU use the same scratch and it keeps the previous call's bits, so every call
 * begins by zeroing the part it will read.  Calls queued on one stream are safe back to back.  Two calls that can
 * run at the same time on one GPU (different streams, different host threads, different contexts of this process)
 * race on it and both results are garbage: serialise them yourself.  The regular workspace path has no such limit. */
#define CC_STATIC_MAX_PAGES (1u << 24)
int32_t cc_dirty_pages_static(int32_t device, const void* cur, const void* shadow, uint64_t bytes, uint32_t page_bytes,
                              uint32_t* d_list, uint32_t list_capacity, uint32_t* d_count, void* stream,
                              int32_t* cuda_error);

/* ============================ BENCH / TEST HOOKS -- not part of the product API ============================
 * Measurement and test instrumentation used by bench.py and tests/ only.  They change no result.  Compiled in by
 * default; build with -DCC_BENCH_HOOKS=0 for a library without them (the worker then answers CC_TASK_TEST_MUTATE
 * with CC_ERR_INVALID).
 * Why the default is ON: the repository builds ONE libconcordia.so and the numbers and parity results it publishes must
 * come from that very binary -- a second, hook-less build would be a library nobody measured.  What the hooks add for a
 * ring client is CC_TASK_TEST_MUTATE, which can flip bytes only inside a region the same process registered through
 * the same context (a ring client already has every pointer).  A deployment that wants them gone sets
 * CC_NVCC_FLAGS=-DCC_BENCH_HOOKS=0 for paper_2606_23521_b200/build.py (bench.py's c5b workload and the worker tests that
 * mutate a region from inside the ring need the hooks and do not run against such a build). */
#ifndef CC_BENCH_HOOKS
#define CC_BENCH_HOOKS 1
#endif
#if CC_BENCH_HOOKS
/* cc_task.kind 4 -- mutate a region from inside the worker, in closed form so that the oracle side can replay it
 * (SURVEY.md 8d C5b): region_id; arg0 = n_mut, arg1 = A (odd), arg2 = h:
 * for j < n_mut: page (j*A + h) mod n_pages, byte (h + j) mod len_p, ^= 0x5A */
#define CC_TASK_TEST_MUTATE 4u
/* If non-NULL, the next host-launched checkpoint / cc_scan_only calls record these cudaEvent_t (passed as void*) on
 * the call's stream right after the discovery (scan) kernel and right after the compaction kernel: per-phase CUDA
 * event timing for bench.py's roofline line.  Pass NULLs to switch it off. */
int32_t cc_trace_events(cc_ctx* ctx, void* ev_after_scan, void* ev_after_compact);
/* Mean host cost of one cc_submit in ns over n CC_TASK_NOP submissions, timed inside the library so that no language
 * binding is in the way (Table 7).  Waits for free slots outside the timed sections and for the last
 * task before returning.  Needs a running worker. */
int32_t cc_measure_submit_cost(cc_ctx* ctx, uint32_t n, double* ns_per_submit);
/* For the comparison with PAPER.md Table 7 (L368-370): mean ns per launch of an empty kernel on `stream`, with a
 * synchronisation after every launch (*ns_sync) and launched back to back with one synchronisation at the end
 * (*ns_batched).  Not while a worker occupies every SM. */
int32_t cc_measure_launch_cost(cc_ctx* ctx, uint32_t n, void* stream, double* ns_sync, double* ns_batched);
#endif /* CC_BENCH_HOOKS */

#ifdef __cplusplus
}
#endif
#endif /* CONCORDIA_H */
