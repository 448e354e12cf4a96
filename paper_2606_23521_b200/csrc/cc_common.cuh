// cc_common.cuh -- device-side data structures and PTX helpers of libconcordia (sm_100a).
// Part of the CUDA path; shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/concordia.h"

typedef uint8_t u8;
typedef uint32_t u32;
typedef uint64_t u64;

#define CC_SEG_BYTES 4096u        // one warp item: 32 lanes x 8 x 16 B
#define CC_SEG_VECS 256u          // 16-byte vectors per segment
#define CC_SEG_POW_MAX 256u       // table of x^(8*4096*m) up to m = 256 (1 MiB of message after a segment)
#define CC_COMPACT_THREADS 256
#define CC_COMPACT_WORDS_PER_THREAD 4
#define CC_COMPACT_TILE_WORDS (CC_COMPACT_THREADS * CC_COMPACT_WORDS_PER_THREAD)   // 1024 words = 32768 pages
#ifndef CC_FUSED_TILE_BYTES
#define CC_FUSED_TILE_BYTES (16u * 1024u)
#endif    // fused pass: one WARP scans (and gathers) this much of the region per ticket
#define CC_FUSED_MAX_TP 32u                  // ... but at most this many pages (the tile's dirty mask is one register)

// Per-region control block in the workspace (device memory).
struct cc_ws_hdr {
    u32 k;              // dirty pages of the last scan
    u32 k_eff;          // records the gather must write (0 on log-full / scan-only)
    int32_t status;     // CC_OK / CC_ERR_LOG_FULL
    u32 ticket;         // compaction tile ticket
    u32 run_id;         // compaction look-back tag
    u32 gather_done;    // warps/blocks finished (last-block pattern)
    u32 fticket;        // fused pass: page-tile ticket (reset by the gather completion, which always follows)
    u32 frun;           // fused pass: look-back tag (bumped by the gather completion)
    u64 W_start;        // log offset at which this checkpoint's records start
    u64 need;           // bytes this checkpoint appends
    u64 t_start_ns;
    u64 epoch;
    u32 inline_done;    // fused pass already wrote the records, headers and shadow: the gather only commits
    u32 commit_k;       // record count that goes into the commit record (= k_eff, or the number of runs)
    u32 n_runs;         // run-length records: runs of the last plan
    u32 pad0;
};

// Device-visible region descriptor.
struct cc_region_dev {
    u8* base;
    u8* shadow;
    u64 bytes;
    u64 n_pages;
    u32 page_bytes;
    u32 region_id;
    u32 spp;            // 4 KiB segments per page = ceil(P / 4096)
    int32_t spp_shift;  // log2(spp) if power of two else -1
    u64 n_words;        // bitmap words
    u32* bitmap;        // n_words (+ padding to a multiple of 4) u32, all zero between calls
    u32* D;             // n_pages u32: ascending dirty list
    u64* rec_state;     // n_pages u64: per-record {done-mask or count : 32 | CRC accumulator : 32}, zero between calls
    u64* lb_status;     // compaction look-back status, one per tile
    u64* flb_status;    // fused pass look-back status, one per page tile
    // run-length records (cc_rle.cuh)
    u32* S;             // bitmap over dirty RANKS: rank i starts a run; same padded size as `bitmap`, zero between calls
    u32* Rfirst;        // n_pages + 1 u32: first rank of run j (and k as a sentinel after the last run)
    u32* Rn;            // n_pages u32: run index of rank i
    u64* run_state;     // n_pages u64: per-run {finished pages : 32 | CRC accumulator : 32}, zero between calls
    cc_ws_hdr* hdr2;    // control block of the ranking pass over S
    u64* lb2;           // its look-back status words
    u32 ftile_pages;    // pages per fused warp tile (~32 KiB of region, 1..32 pages)
    u32 n_ftiles;
    u32* latest;        // n_pages u32: applier last-wins table, all zero between calls
    cc_ws_hdr* hdr;
    u32 crc_init_full;  // 0xFFFFFFFF * x^(8*P): the CRC init term of a full page
    u32 crc_init_tail;  // same for the (possibly short) last page
};

struct cc_log_dev {
    u8* buf;
    u64 capacity;
    u64 W;                  // running write offset (device-resident so that async calls chain)
    u64* committed_off;     // host-visible published offset (may be null)
    u64 gen;                // number of resets so far: the log's generation
    u64* pub;               // library-owned pinned word (gen << 48 | committed offset) that the drainer thread follows
};
#define CC_PUB_SHIFT 48

// Applier tables (in the attached scratch).
struct cc_rec {             // 32 bytes
    u64 off;                // offset of the record header in the log
    u32 page_idx;
    u32 len;
    u32 crc;
    u32 slot;               // region slot
    u32 epoch_idx;
    u32 pad;
};
struct cc_epoch_ent {       // 32 bytes
    u64 off_after;          // log offset right after the epoch's commit record
    u64 epoch_no;           // the epoch number its commit record carries
    u32 rec_end;            // records [.., rec_end) belong to epochs <= this one
    u32 slot;               // region slot of its records (0xFFFFFFFF: an empty epoch)
    u32 pending;            // its record count
    u32 pad;
};
struct cc_apply_state {
    u32 n_recs;
    u32 n_epochs;
    u32 struct_fail;        // 1 if the parse stopped on a failed structural check
    u32 scratch_overflow;
    u32 first_bad_rec;      // min index of a record failing CRC (init 0xFFFFFFFF)
    u32 validate_done;
    u32 n_commit_recs;      // records in applied epochs
    u32 n_commit_epochs;
    u64 consumed;
    u64 t_start_ns;
    int32_t status;
    u32 final_done;
};

// Log compactor state (cc_compactor.cuh).
struct cc_compactor_state {
    u32 region_last[CC_MAX_REGIONS];    // 1 + index of the last input epoch that touched the region (0: none)
    u64 bytes_out;
    u64 n_out;
    int32_t status;
    u32 n_regions_out;
};

// Multi-region boundary checkpoint state (cc_batch.cuh).
struct cc_batch_state {
    u64 W_final;
    u64 k_total;
    u64 bytes_total;
    u64 t_start_ns;
    u64 epoch;
    int32_t status;         // CC_OK or the status of the first (lowest id) region that failed
    u32 n_active;           // regions taking part (those with a shadow)
    u32 done;               // regions whose commit record is in place
    u32 pad;
};

struct cc_parse_ctl {                    // control block of the parallel parse (cc_apply_parse.cuh)
    u32 n_raw;                           // candidate search: hits appended so far (reset by the walk phase)
    u32 n_cand;                          // candidates on the ordered list
    u32 cand_overflow;                   // reset by the validation's resolver
    u32 need_serial;                     // the serial parser must redo the parse (reset by the validation's resolver)
    u32 wticket;                         // walk: span ticket (reset by the validation phase)
    u32 pad[3];
};

struct alignas(16) cc_crc_tables {
    u32 t0[256];            // byte table of the reflected polynomial
    u32 t0k[3][256];        // t0k[k-1]: the same for a byte followed by k zero bytes (slicing-by-4, cc_crc_smem4)
    alignas(16) u32 s512[4][256];       // multiply by x^(8*512) mod G, one table per register byte
    u32 lane_mul[32];       // x^(8*16*(31-lane))
    u32 seg_mul[CC_SEG_POW_MAX + 1];   // x^(8*4096*m), m = 0..CC_SEG_POW_MAX
    u32 xp[48];             // x^(8*2^j), j = 0..47
    alignas(16) u32 lane_nib[8 * 16 * 32];  // (v << 4n) * lane_mul[l] at [(n*16 + v)*32 + l]
    u32 seg_pow[(CC_SEG_POW_MAX + 1) * 32];   // seg_mul[m] * x^i at [m*32 + i]
};

struct cc_dev {
    cc_region_dev regions[CC_MAX_REGIONS];
    u32 region_used[CC_MAX_REGIONS];
    cc_log_dev log;
    cc_crc_tables crc;
    // applier
    cc_rec* recs;
    cc_epoch_ent* epochs;
    u64 max_records;
    cc_apply_state apply;
    cc_parse_ctl parse;
    cc_compactor_state compactor;
    cc_batch_state batch;
    // grid barrier + worker doorbell
    u32 bar_count;
    u32 bar_gen;
    u64 doorbell;
    alignas(16) cc_task cur_task;
    u32 worker_exit;
    u64 trace[32];          // -DCC_TRACE_ON=1 probe builds only: %globaltimer stamps of the phases
};

#ifndef CC_TRACE_ON
#define CC_TRACE_ON 0
#endif
#if CC_TRACE_ON
#define CC_TRACE(dev, i) do { (dev)->trace[i] = globaltimer_ns(); } while (0)
#define CC_TRACE_MAX(dev, i, lane) do { if ((lane) == 0) atomicMax(reinterpret_cast<unsigned long long*>(&(dev)->trace[i]), (unsigned long long)globaltimer_ns()); } while (0)
#else
#define CC_TRACE(dev, i) do { } while (0)
#define CC_TRACE_MAX(dev, i, lane) do { } while (0)
#endif

// ------------------------------------------------------------------ PTX helpers --

// Streaming 16-byte load of region / shadow bytes.  COHERENT (no .nc): the same device code runs inside the
// persistent worker, where base and shadow are rewritten by earlier tasks (gather, restore, the application's
// kernels) while the kernel stays resident -- PTX allows .nc only for data that is read-only for the kernel's
// whole lifetime.  L1::no_allocate keeps the stream out of L1 either way.  -DCC_LD_NC=1 builds the
// non-coherent variant for an A/B measurement (profiles/r02_ld_nc.md: no bandwidth difference).
#ifndef CC_LD_NC
#define CC_LD_NC 0
#endif
__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
    uint4 r;
#if CC_LD_NC
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
#else
    asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
#endif
    return r;
}
// Plain (coherent) 16-byte load: log buffers may live in host memory and may have been
// written by another kernel moments ago; no non-coherent path.
__device__ __forceinline__ uint4 ld_v4(const uint4* p) {
    uint4 r;
    asm volatile("ld.global.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(uint4* p, const uint4& v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
// Programmatic dependent launch (sm_90+): a kernel launched with the programmatic-stream-serialization attribute may
// start while its predecessor in the stream is still running; it must execute cc_pdl_wait() before it touches anything
// the predecessor writes (no-op when launched normally).  cc_pdl_trigger() in the predecessor lets the dependent grid
// be scheduled as soon as SM resources free up.  OFF by default (-DCC_PDL=1 builds with it): measured with the calls
// queued ahead of the GPU, plain stream order is faster (C5a replay 0.382 vs 0.400 ms, C1 checkpoint 51.9 vs 53.9 us).
#ifndef CC_PDL
#define CC_PDL 0
#endif
__device__ __forceinline__ void cc_pdl_wait() {
#if CC_PDL
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
}
__device__ __forceinline__ void cc_pdl_trigger() {
#if CC_PDL
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
}
__device__ __forceinline__ u64 globaltimer_ns() {
    u64 t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ u64 ld_acquire_gpu_u64(const u64* p) {
    u64 v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu_u64(u64* p, u64 v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
// Relaxed gpu-scope accesses: for words whose VALUE is the whole message (look-back status words), so that
// publishing them does not have to wait for the thread's earlier (possibly host-link) stores.
__device__ __forceinline__ u64 ld_relaxed_gpu_u64(const u64* p) {
    u64 v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_gpu_u64(u64* p, u64 v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ u32 ld_acquire_gpu_u32(const u32* p) {
    u32 v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ u64 ld_acquire_sys_u64(const u64* p) {
    u64 v;
    asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_sys_u64(u64* p, u64 v) {
    asm volatile("st.release.sys.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint4 ld_relaxed_sys_v4(const void* p) {
    uint4 r;
    asm volatile("ld.relaxed.sys.global.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st_relaxed_sys_u64(u64* p, u64 v) {
    asm volatile("st.relaxed.sys.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ u32 ld_relaxed_sys_u32(const u32* p) {
    u32 v;
    asm volatile("ld.relaxed.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// One thread, after the CALLER has executed __threadfence_system() behind the commit record ("a commit
// marker publishes the epoch only after all bytes are visible") and whatever else must be visible first: advance the
// write offset and publish the committed offset -- to the caller's word and to the library's own (generation-tagged)
// word -- with plain system-scope stores (every release store would be another full fence, ~2 us each with host-memory
// stores in flight).
__device__ __forceinline__ void cc_log_publish_fenced(cc_log_dev* log, u64 W_after) {
    if (log->committed_off) st_relaxed_sys_u64(log->committed_off, W_after);
    if (log->pub) st_relaxed_sys_u64(log->pub, (log->gen << CC_PUB_SHIFT) | W_after);
    log->W = W_after;
}
// W := 0: a new generation of the log (cc_log_reset*, CC_TASK_LOG_RESET).  One fence, then the two words.
__device__ __forceinline__ void cc_log_rewind(cc_log_dev* log) {
    log->gen = log->gen + 1;
    log->W = 0;
    __threadfence_system();
    if (log->committed_off) st_relaxed_sys_u64(log->committed_off, 0ull);
    if (log->pub) st_relaxed_sys_u64(log->pub, log->gen << CC_PUB_SHIFT);
}

__device__ __forceinline__ u64 page_len_dev(const cc_region_dev& r, u64 p) {
    u64 rest = r.bytes - p * (u64)r.page_bytes;
    return rest < r.page_bytes ? rest : (u64)r.page_bytes;
}

// Virtual grid: the same device code runs as a host-launched kernel (blockIdx/gridDim) and
// inside the persistent worker.
struct cc_grid {
    u32 block, nblocks;
    __device__ __forceinline__ u32 warp() const { return block * (blockDim.x >> 5) + (threadIdx.x >> 5); }
    __device__ __forceinline__ u32 nwarps() const { return nblocks * (blockDim.x >> 5); }
};
__device__ __forceinline__ cc_grid cc_hw_grid() { return cc_grid{blockIdx.x, gridDim.x}; }
