// concordia.cu -- libconcordia.so: kernels (thin __global__ wrappers over the device phases)
// and the C ABI of include/concordia.h.  sm_100a only.  No CPU fallback: every step of the path
// runs in the kernels below; the host code only validates arguments, keeps the region table and
// launches.
#include <atomic>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <mutex>
#include <thread>
#include <time.h>

#include "cc_common.cuh"
#include "cc_crc.cuh"
#include "cc_ckpt.cuh"
#include "cc_mark.cuh"
#include "cc_fused.cuh"
#include "cc_pass.cuh"
#include "cc_small.cuh"
#include "cc_tasks.cuh"
#include "cc_rle.cuh"
#include "cc_apply.cuh"
#include "cc_compactor.cuh"
#include "cc_batch.cuh"
#include "cc_worker.cuh"

static_assert(sizeof(cc_result) == 64, "cc_result must be 64 bytes");
static_assert(sizeof(cc_task) == 64, "cc_task must be 64 bytes");
static_assert(sizeof(cc_rec) == 32, "cc_rec must be 32 bytes");

// ------------------------------------------------------------------------ kernels --

#ifndef CC_PASS_LAZY_CRC
#define CC_PASS_LAZY_CRC 0          // 1: A/B of the lazily filled CRC tables
#endif

#define CC_SCAN_THREADS 256
#define CC_SMALL_TAIL_MAX_BYTES (1ull << 30)         // phases path: up to this region size the compaction kernel is replaced by in-block ranking
#define CC_PASS_AUTO_MIN_BYTES (128ull << 20)        // CC_PATH_AUTO: single pass for pinned host logs from this region size on
#define CC_GATHER_THREADS 256
#define CC_APPLY_THREADS 256
#define CC_PARSE_THREADS 1024

__global__ void __launch_bounds__(CC_SCAN_THREADS) cc_scan_kernel(cc_dev* dev, const __grid_constant__ cc_region_dev rg) {
    cc_pdl_trigger();                       // the compaction (and behind it the gather) may queue up behind this grid
    if (blockIdx.x == 0 && threadIdx.x == 0) CC_TRACE(dev, 0);
    cc_scan_phase<8>(rg, cc_hw_grid());
    if (blockIdx.x == 0 && threadIdx.x == 0) CC_TRACE(dev, 1);
}

__global__ void __launch_bounds__(CC_COMPACT_THREADS) cc_compact_kernel(cc_dev* dev, const __grid_constant__ cc_region_dev rg, u32 mode, u64 epoch,
                                                                        cc_result* out) {
    cc_pdl_trigger();
    cc_pdl_wait();                          // the bitmap is complete
    if (blockIdx.x == 0 && threadIdx.x == 0) CC_TRACE(dev, 2);
    cc_compact_phase(rg, &dev->log, mode, epoch, out);
    if (blockIdx.x == 0 && threadIdx.x == 0) CC_TRACE(dev, 3);
}

#ifndef CC_GATHER_MIN_BLOCKS
#define CC_GATHER_MIN_BLOCKS 4
#endif
__global__ void __launch_bounds__(CC_GATHER_THREADS, CC_GATHER_MIN_BLOCKS) cc_gather_kernel(cc_dev* dev, const __grid_constant__ cc_region_dev rg, cc_result* out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (blockIdx.x == 0 && threadIdx.x == 0) CC_TRACE(dev, 4);
    cc_crc_smem* cs = reinterpret_cast<cc_crc_smem*>(smem_raw);
#if CC_PDL
    // the CRC tables do not depend on the plan: filled while the compaction is still running (programmatic dependent
    // launch), then wait for the plan
    cc_crc_smem_init(cs, &dev->crc);
    cc_pdl_wait();
    cc_gather_phase(rg, dev, cs, cc_hw_grid(), out, CC_TASK_DELTA_CKPT, false);
#else
    // plain stream order: only the blocks that have records to write fill the tables (a sparse checkpoint keeps 20 of
    // 592 blocks busy; the other 572 fetching 52 KiB each out of L2 delayed those 20)
    cc_gather_phase(rg, dev, cs, cc_hw_grid(), out, CC_TASK_DELTA_CKPT, true);
#endif
}

// The whole checkpoint of one region in ONE launch (cc_pass.cuh).  Cooperative: when the worst case does not fit
// behind the write offset the classic phases run instead, separated by grid barriers.
__global__ void __launch_bounds__(CC_GATHER_THREADS, 4) cc_pass_kernel(cc_dev* dev, const __grid_constant__ cc_region_dev rg, cc_pass_args a, cc_result* out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cc_crc_smem* cs = reinterpret_cast<cc_crc_smem*>(smem_raw);
    __shared__ u32 s_crc_state, s_warps_left;
    const cc_region_dev& r = rg;
    const cc_grid g = cc_hw_grid();
    if (threadIdx.x == 0) { s_crc_state = 0; s_warps_left = blockDim.x >> 5; }
    if (g.block == 0 && threadIdx.x == 0) { r.hdr->t_start_ns = globaltimer_ns(); CC_TRACE(dev, 10); }
    __syncthreads();
    const u64 W0 = dev->log.W;
    const bool inline_ok = dev->log.buf != nullptr && W0 + cc_pass_worst_bytes(r) <= dev->log.capacity;
    if (inline_ok) {
        const u32 lane = threadIdx.x & 31u;
#if !CC_PASS_LAZY_CRC
        // the CRC tables, by the whole block at once (~2 us).  (Filled lazily by the first warp that needs them, that warp
        // alone takes ~30 us over it -- on the critical path of every call that has a dirty page.)
        cc_crc_smem_init(cs, &dev->crc);
        if (threadIdx.x == 0) s_crc_state = 2u;
        __syncthreads();
#endif
        const u32 TP = cc_pass_tile_pages(r, a.run_pages, g.nwarps());
        const bool wrote = cc_pass_tiles(r, dev, cs, &s_crc_state, a, TP, W0, g);
        if (g.block == 0 && threadIdx.x == 0) CC_TRACE(dev, 11);
        if (cc_pass_leave(r.hdr, &s_warps_left, wrote, g.nblocks, lane)) {
            if (lane == 0) CC_TRACE(dev, 12);
            cc_pass_commit(r, dev, out, a.kind, lane);
            if (lane == 0) CC_TRACE(dev, 13);
        }
        return;
    }
    u32 gen = ld_acquire_gpu_u32(&dev->bar_gen);
    cc_classic_checkpoint(dev, r, cs, a, g, gen, out, true);
}

// The low-latency checkpoint of a small region in ONE launch (cc_small.cuh).  Cooperative: one grid-wide rendezvous.
__global__ void __launch_bounds__(CC_GATHER_THREADS, 4) cc_small_kernel(cc_dev* dev, const __grid_constant__ cc_region_dev rg, u64 epoch, cc_result* out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ cc_small_smem s_small;
    u32 gen = ld_acquire_gpu_u32(&dev->bar_gen);
    cc_small_checkpoint(dev, rg, reinterpret_cast<cc_crc_smem*>(smem_raw), &s_small, epoch, CC_TASK_DELTA_CKPT,
                        cc_hw_grid(), gen, out, true);
}

// The same path as TWO launches for host-launched calls: cc_scan_kernel at its own occupancy (47 resident warps per SM),
// then rank + write + commit -- no compaction kernel, no dirty list to wait for (a plain launch: no block waits on another).
__global__ void __launch_bounds__(CC_GATHER_THREADS, 4) cc_small_tail_kernel(cc_dev* dev, const __grid_constant__ cc_region_dev rg, u64 epoch,
                                                                            cc_result* out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ cc_small_smem s_small;
    if (blockIdx.x == 0 && threadIdx.x == 0) CC_TRACE(dev, 11);
    cc_small_tail(dev, rg, reinterpret_cast<cc_crc_smem*>(smem_raw), &s_small, epoch, CC_TASK_DELTA_CKPT, cc_hw_grid(), out, false);
}

__global__ void __launch_bounds__(256) cc_snapshot_plan_kernel(const cc_dev* dev, const __grid_constant__ cc_region_dev rg, u64 epoch) {
    cc_snapshot_plan_phase(rg, &dev->log, epoch, cc_hw_grid());
}

// log compactor (cc_compactor.cuh)
__global__ void __launch_bounds__(CC_APPLY_THREADS) cc_compactor_mark_kernel(cc_dev* dev, cc_apply_tabs tabs) {
    cc_compactor_mark_phase(dev, tabs, cc_hw_grid());
}
__global__ void __launch_bounds__(CC_COMPACT_THREADS) cc_compactor_rank_kernel(cc_dev* dev) { cc_compactor_rank_phase(dev); }
__global__ void __launch_bounds__(CC_MAX_REGIONS) cc_compactor_plan_kernel(cc_dev* dev, u64 out_capacity) { cc_compactor_plan_phase(dev, out_capacity); }
__global__ void __launch_bounds__(CC_APPLY_THREADS) cc_compactor_copy_kernel(cc_dev* dev, cc_apply_tabs tabs, const u8* in, u8* out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cc_crc_smem* cs = reinterpret_cast<cc_crc_smem*>(smem_raw);
    cc_crc_smem_init(cs, &dev->crc);
    cc_compactor_copy_phase(dev, tabs, cs, in, out, cc_hw_grid());
}
__global__ void __launch_bounds__(CC_APPLY_THREADS) cc_compactor_cleanup_kernel(cc_dev* dev, cc_apply_tabs tabs, cc_result* out) {
    cc_compactor_cleanup_phase(dev, tabs, cc_hw_grid(), out, CC_TASK_COMPACT_LOG);
}

// run-length records (cc_rle.cuh)
__global__ void __launch_bounds__(256) cc_rle_starts_kernel(const cc_dev* dev, const __grid_constant__ cc_region_dev rg, u32 run_pages) {
    cc_rle_starts_phase(rg, run_pages, cc_hw_grid());
}
__global__ void __launch_bounds__(CC_COMPACT_THREADS) cc_rle_rank_kernel(const cc_dev* dev, const __grid_constant__ cc_region_dev rg) {
    cc_rle_rank_phase(rg, &dev->log);
}
__global__ void __launch_bounds__(256) cc_rle_plan_kernel(const cc_dev* dev, const __grid_constant__ cc_region_dev rg, u64 epoch) {
    cc_rle_plan_phase(rg, &dev->log, epoch, cc_hw_grid());
}
__global__ void __launch_bounds__(CC_GATHER_THREADS, 4) cc_rle_gather_kernel(cc_dev* dev, const __grid_constant__ cc_region_dev rg, cc_result* out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cc_rle_gather_phase(rg, dev, reinterpret_cast<cc_crc_smem*>(smem_raw), cc_hw_grid(), out,
                        CC_TASK_DELTA_CKPT, true);
}

// one boundary, all regions (cc_batch.cuh)
__global__ void __launch_bounds__(CC_SCAN_THREADS) cc_batch_scan_kernel(cc_dev* dev) {
    __shared__ cc_batch_tab tab;
    cc_batch_scan_phase(dev, &tab, cc_hw_grid());
}
__global__ void __launch_bounds__(CC_COMPACT_THREADS) cc_batch_rank_kernel(cc_dev* dev, u64 epoch) {
    cc_batch_rank_phase(dev, epoch, cc_hw_grid());
}
__global__ void __launch_bounds__(CC_MAX_REGIONS) cc_batch_plan_kernel(cc_dev* dev, u64 epoch) { cc_batch_plan_phase(dev, epoch); }
__global__ void __launch_bounds__(CC_GATHER_THREADS, 4) cc_batch_gather_kernel(cc_dev* dev, cc_result* out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cc_crc_smem* cs = reinterpret_cast<cc_crc_smem*>(smem_raw);
    __shared__ cc_batch_tab tab;
    cc_crc_smem_init(cs, &dev->crc);
    cc_batch_gather_phase(dev, cs, &tab, cc_hw_grid(), out, CC_TASK_CKPT_ALL);
}

// cc_checkpoint_all_rle: the per-region calls have run (stream order); one thread sums their plans up into the result
struct cc_slot_list { int n; int slot[CC_MAX_REGIONS]; };
__global__ void cc_batch_collect_kernel(cc_dev* dev, cc_slot_list L, u64 epoch, u64 t_start_ns, cc_result* out) {
    if (!out) return;
    u64 k = 0, bytes = 0;
    int32_t st = CC_OK;
    for (int i = 0; i < L.n; i++) {                    // ascending region_id
        const cc_ws_hdr* h = dev->regions[L.slot[i]].hdr;
        k += h->k;
        bytes += h->need;
        if (st == CC_OK && h->status != CC_OK) st = h->status;
    }
    out->n_dirty = k;
    out->bytes = bytes;
    out->log_offset_after = dev->log.W;
    out->epoch = epoch;
    out->status = st;
    out->flags = CC_TASK_CKPT_ALL;
    out->t_start_ns = L.n ? dev->regions[L.slot[0]].hdr->t_start_ns : t_start_ns;
    out->t_end_ns = globaltimer_ns();
    __threadfence_system();
    st_relaxed_sys_u64(&out->seq_done, 1ull);
}

// allocator-aware discovery (cc_mark.cuh)
__global__ void __launch_bounds__(256) cc_mark_load_kernel(const cc_dev* dev, const __grid_constant__ cc_region_dev rg, const u32* marks) {
    cc_mark_load_phase(rg, marks, cc_hw_grid());
}
__global__ void __launch_bounds__(256) cc_mark_versions_kernel(const cc_dev* dev, const __grid_constant__ cc_region_dev rg, const u64* version,
                                                               const u64* committed) {
    cc_mark_versions_phase(rg, version, committed, cc_hw_grid());
}
__global__ void __launch_bounds__(CC_SCAN_THREADS) cc_mark_verify_kernel(const cc_dev* dev, const __grid_constant__ cc_region_dev rg) {
    cc_mark_verify_phase(rg, cc_hw_grid());
}
__global__ void __launch_bounds__(256) cc_mark_finish_kernel(const cc_dev* dev, const __grid_constant__ cc_region_dev rg, u32* marks_to_clear,
                                                             const u64* version, u64* committed) {
    cc_mark_finish_phase(rg, marks_to_clear, version, committed, cc_hw_grid());
}

// parse: candidate commit records (whole log, grid-wide) -> epoch walks (one block per epoch, chained by look-back)
// -> the one-block serial walk, which returns at once unless the parallel parse asked for it
// (In a -DCC_PDL=1 build every launch of the chain carries the programmatic-serialization attribute: a kernel lets its
// successor be scheduled at once, cc_pdl_trigger, and waits for its predecessor's results itself, cc_pdl_wait.  Off by
// default: measured slower than plain stream order, see cc_common.cuh.)
__global__ void __launch_bounds__(CC_CAND_THREADS) cc_apply_cand_kernel(cc_dev* dev, cc_apply_tabs tabs, const u8* log, u64 n) {
    cc_pdl_trigger();                           // (launched normally: ordered behind whatever the stream held before)
    cc_parse_cand_phase(dev, &dev->parse, tabs.cand_raw, tabs.max_records, log, n, cc_hw_grid());
}
__global__ void __launch_bounds__(CC_SORT_THREADS) cc_apply_sort_kernel(cc_dev* dev, cc_apply_tabs tabs) {
    cc_pdl_trigger();
    cc_pdl_wait();
    cc_parse_sort_phase(&dev->parse, tabs.cand_raw, tabs.cand, tabs.span_status, tabs.max_records, cc_hw_grid());
}
__global__ void __launch_bounds__(CC_WALK_THREADS) cc_apply_walk_kernel(cc_dev* dev, cc_apply_tabs tabs, const u8* log, u64 n) {
    cc_pdl_trigger();
    cc_pdl_wait();
    cc_parse_walk_phase(dev, &dev->parse, tabs, log, n, blockIdx.x == 0);
}
__global__ void __launch_bounds__(CC_PARSE_THREADS) cc_apply_parse_kernel(cc_dev* dev, cc_apply_tabs tabs, const u8* log, u64 n) {
    cc_pdl_trigger();
    cc_pdl_wait();
    cc_apply_parse_phase(dev, tabs, log, n, false);
}

// The validation is bound by instruction issue: it runs the slicing-by-4 CRC (cc_crc_smem4: 128 KiB of lane-replicated
// tables, 2.5 instead of 4.5 instructions per payload byte and lane) as ONE block of 1,024 threads per SM.
#define CC_VALIDATE_THREADS 1024
__global__ void __launch_bounds__(CC_VALIDATE_THREADS, 1) cc_apply_validate_kernel(cc_dev* dev, cc_apply_tabs tabs, const u8* log) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cc_crc_smem4* cs = reinterpret_cast<cc_crc_smem4*>(smem_raw);
    cc_pdl_trigger();
    cc_crc_smem_init(cs, &dev->crc);            // (does not depend on the parse)
    cc_pdl_wait();
    cc_apply_validate_phase(dev, tabs, cs, log, cc_hw_grid(), false);
}

__global__ void __launch_bounds__(CC_APPLY_THREADS) cc_apply_latest_kernel(cc_dev* dev, cc_apply_tabs tabs) {
    cc_pdl_trigger();
    cc_pdl_wait();
    cc_apply_latest_phase(dev, tabs, cc_hw_grid());
}

__global__ void __launch_bounds__(CC_APPLY_THREADS) cc_apply_scatter_kernel(cc_dev* dev, cc_apply_tabs tabs, const u8* log) {
    cc_pdl_trigger();
    cc_pdl_wait();
    cc_apply_scatter_phase(dev, tabs, log, cc_hw_grid());
}

__global__ void __launch_bounds__(CC_APPLY_THREADS) cc_apply_cleanup_kernel(cc_dev* dev, cc_apply_tabs tabs, cc_result* out) {
    cc_pdl_wait();
    cc_apply_cleanup_phase(dev, tabs, cc_hw_grid(), out, CC_TASK_RESTORE);
}

// --------------------------------------------------------------------- host context --

struct cc_host_region {
    bool used;
    cc_region_desc desc;
    cc_region_dev dev;
};

struct cc_ctx {
    int device;
    cc_config cfg;
    int sm_count;
    cc_dev* d_dev;
    cudaStream_t internal;
    cc_host_region regions[CC_MAX_REGIONS];
    bool log_attached;
    bool log_is_host;           // the attached log is pinned host memory (records cross the host link)
    uint64_t* committed_off;    // the caller's published-offset word (may be null)
    void* log_buf;              // the attached log (device or pinned host)
    uint64_t log_capacity;
    // host mirror of a device-resident log, filled by the copy engine (cc_log_mirror_attach / cc_log_drain)
    void* mirror;
    uint64_t mirror_capacity;
    uint64_t* mirror_committed;
    uint64_t drained;
    cudaEvent_t drain_ev;
    // library-side drainer (cc_log_drain_start / _stop): a host thread that follows the published offset
    std::thread* drainer;
    std::atomic<uint32_t> drainer_stop;
    std::atomic<uint64_t> drainer_gen;      // generation the thread is draining
    std::atomic<uint64_t> drainer_landed;   // bytes of that generation whose copies have completed
    std::atomic<int32_t> drainer_status;
    cudaStream_t drainer_stream;
    cc_apply_tabs tabs;
    bool apply_attached;
    void* stage;                // optional device staging buffer for host-resident logs (cc_apply_stage_attach)
    uint64_t stage_bytes;
    uint64_t stage_used = 0, stage_bypassed = 0;   // host-resident logs copied into the staging buffer / read in place although one is attached
    int last_cuda;
    uint64_t launches;
    int scan_bps, gather_bps, validate_bps, fused_bps, small_bps, cand_bps;     // blocks per SM from the occupancy API
    // ring + worker (pinned host)
    cc_task* ring_slots;
    cc_result* ring_results;
    u64* ring_words;            // [0] tail, [8] completed, [16] heartbeat (one cache line apart)
    u64 submitted;
    std::atomic<uint32_t> in_submit;   // single-producer guard of cc_submit
    bool worker_running;
    cudaStream_t worker_stream;
    cudaEvent_t worker_done;
    u32 worker_blocks_used;
    cudaEvent_t ev_after_scan, ev_after_compact;
};

#define CC_CUDA(ctx, call)                                     \
    do {                                                       \
        cudaError_t e__ = (call);                              \
        if (e__ != cudaSuccess) {                              \
            (ctx)->last_cuda = (int)e__;                       \
            return CC_ERR_CUDA;                                \
        }                                                      \
    } while (0)

static const u8* stage_log(cc_ctx* ctx, const void* log, uint64_t nbytes, cudaStream_t st);

// The host-launched data-path calls share the per-region control blocks, the log write offset and the applier
// tables with the resident worker: while it runs they are refused (submit the matching task instead).
#define CC_NO_WORKER(ctx)                                      \
    do {                                                       \
        if ((ctx)->worker_running) return CC_ERR_WORKER;       \
    } while (0)

static inline uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

static int find_slot(cc_ctx* ctx, uint32_t id) {
    for (int s = 0; s < CC_MAX_REGIONS; s++)
        if (ctx->regions[s].used && ctx->regions[s].desc.region_id == id) return s;
    return -1;
}

struct cc_ws_layout {
    uint64_t hdr, bitmap, D, rec_state, latest, lb, flb, S, Rfirst, Rn, run_state, hdr2, lb2, total;
    uint64_t n_pages, n_words, n_tiles, ftile_pages, n_ftiles;
};

static bool ws_layout(uint64_t bytes, uint32_t P, cc_ws_layout* L) {
    if (P == 0 || (P & 15u) || bytes == 0 || (bytes & 15ull)) return false;
    uint64_t n_pages = (bytes + P - 1) / P;
    if (n_pages > (1ull << 31)) return false;
    L->n_pages = n_pages;
    L->n_words = (n_pages + 31) / 32;
    L->n_tiles = (L->n_words + CC_COMPACT_TILE_WORDS - 1) / CC_COMPACT_TILE_WORDS;
    uint64_t o = 0;
    L->hdr = o; o += 256;
    L->bitmap = o; o += align_up(L->n_tiles * CC_COMPACT_TILE_WORDS * 4, 256);
    L->D = o; o += align_up(n_pages * 4, 256);
    L->rec_state = o; o += align_up(n_pages * 8, 256);
    L->latest = o; o += align_up(n_pages * 4, 256);
    L->lb = o; o += align_up(L->n_tiles * 8, 256);
    // single pass (cc_pass.cuh): one look-back word per warp tile, at most CC_PASS_MAX_TILES tiles (pages and records)
    L->n_ftiles = n_pages < CC_PASS_MAX_TILES ? n_pages : CC_PASS_MAX_TILES;
    L->ftile_pages = 0;
    L->flb = o; o += align_up((L->n_ftiles + 32) * 8, 256);
    // run-length records (cc_rle.cuh)
    L->S = o; o += align_up(L->n_tiles * CC_COMPACT_TILE_WORDS * 4, 256);
    L->Rfirst = o; o += align_up((n_pages + 1) * 4, 256);
    L->Rn = o; o += align_up(n_pages * 4, 256);
    L->run_state = o; o += align_up(n_pages * 8, 256);
    L->hdr2 = o; o += 256;
    L->lb2 = o; o += align_up(((L->n_ftiles > L->n_tiles ? L->n_ftiles : L->n_tiles) + 32) * 8, 256);
    L->total = o;
    return true;
}

// ------------------------------------------------------------------------ lifecycle --

extern "C" int32_t cc_init(cc_ctx** out, int32_t device, const cc_config* cfg) {
    if (!out) return CC_ERR_INVALID;
    *out = nullptr;
    cc_ctx* ctx = new (std::nothrow) cc_ctx();       // value-initialised: every field zero
    if (!ctx) return CC_ERR_INVALID;
    ctx->device = device;
    if (cfg) ctx->cfg = *cfg;
    if (ctx->cfg.ring_capacity == 0) ctx->cfg.ring_capacity = 256;
    if (ctx->cfg.worker_threads == 0) ctx->cfg.worker_threads = CC_WORKER_MAX_THREADS;
    if (ctx->cfg.backoff_ns == 0) ctx->cfg.backoff_ns = 500;
    if (ctx->cfg.max_lifetime_ns == 0) ctx->cfg.max_lifetime_ns = 600ull * 1000000000ull;
    const uint32_t cap = ctx->cfg.ring_capacity;
    if ((cap & (cap - 1)) || ctx->cfg.worker_threads > CC_WORKER_MAX_THREADS || (ctx->cfg.worker_threads & 31u) ||
        ctx->cfg.worker_threads < CC_COMPACT_THREADS) {
        delete ctx;
        return CC_ERR_INVALID;
    }
    cudaError_t e = cudaSetDevice(device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, device);
    if (e == cudaSuccess && prop.major < 10) e = cudaErrorNoKernelImageForDevice;   // sm_100a code only
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_dev, sizeof(cc_dev));
    if (e != cudaSuccess) {
        fprintf(stderr, "libconcordia: cc_init failed: %s (no CPU fallback exists)\n", cudaGetErrorString(e));
        delete ctx;
        return CC_ERR_CUDA;
    }
    ctx->sm_count = prop.multiProcessorCount;
    cc_dev* h = (cc_dev*)calloc(1, sizeof(cc_dev));
    cc_crc_build_tables(&h->crc);
    e = cudaMemcpy(ctx->d_dev, h, sizeof(cc_dev), cudaMemcpyHostToDevice);
    free(h);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->internal, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->worker_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->worker_done, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_gather_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_rle_gather_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_compactor_copy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_batch_gather_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_pass_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->fused_bps, cc_pass_kernel, CC_GATHER_THREADS, sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_small_tail_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->small_bps, cc_small_kernel, CC_GATHER_THREADS, sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_apply_validate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem4));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cc_worker_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->scan_bps, cc_scan_kernel, CC_SCAN_THREADS, 0);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->gather_bps, cc_gather_kernel, CC_GATHER_THREADS, sizeof(cc_crc_smem));
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->cand_bps, cc_apply_cand_kernel, CC_CAND_THREADS, 0);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->validate_bps, cc_apply_validate_kernel, CC_VALIDATE_THREADS, sizeof(cc_crc_smem4));
    // ring + completion slots + control words: pinned, device-mapped host memory
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&ctx->ring_slots, (size_t)cap * sizeof(cc_task), cudaHostAllocMapped | cudaHostAllocPortable);
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&ctx->ring_results, (size_t)cap * sizeof(cc_result), cudaHostAllocMapped | cudaHostAllocPortable);
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&ctx->ring_words, 256, cudaHostAllocMapped | cudaHostAllocPortable);
    if (e != cudaSuccess) {
        fprintf(stderr, "libconcordia: cc_init failed: %s\n", cudaGetErrorString(e));
        ctx->last_cuda = (int)e;
        cc_shutdown(ctx);
        return CC_ERR_CUDA;
    }
    memset(ctx->ring_slots, 0, (size_t)cap * sizeof(cc_task));
    memset(ctx->ring_results, 0, (size_t)cap * sizeof(cc_result));
    memset(ctx->ring_words, 0, 256);
    if (ctx->scan_bps < 1) ctx->scan_bps = 1;
    if (ctx->gather_bps < 1) ctx->gather_bps = 1;
    if (ctx->validate_bps < 1) ctx->validate_bps = 1;
    if (ctx->fused_bps < 1) ctx->fused_bps = 1;
    if (ctx->small_bps < 1) ctx->small_bps = 1;
    if (ctx->cand_bps < 1) ctx->cand_bps = 1;
    *out = ctx;
    return CC_OK;
}

extern "C" int32_t cc_shutdown(cc_ctx* ctx) {
    if (!ctx) return CC_ERR_INVALID;
    cudaSetDevice(ctx->device);
    int32_t rc = CC_OK;
    if (ctx->drainer) cc_log_drain_stop(ctx);
    if (ctx->worker_running) rc = cc_worker_stop(ctx);
    if (rc == CC_ERR_TIMEOUT) return rc;    // the kernel may still be resident and reads *ctx's ring: leak rather than free under it
    if (rc == CC_OK) {   // never free under a resident kernel
        if (ctx->d_dev) cudaFree(ctx->d_dev);
        if (ctx->ring_slots) cudaFreeHost(ctx->ring_slots);
        if (ctx->ring_results) cudaFreeHost(ctx->ring_results);
        if (ctx->ring_words) cudaFreeHost(ctx->ring_words);
        if (ctx->internal) cudaStreamDestroy(ctx->internal);
        if (ctx->worker_stream) cudaStreamDestroy(ctx->worker_stream);
        if (ctx->worker_done) cudaEventDestroy(ctx->worker_done);
        if (ctx->drain_ev) cudaEventDestroy(ctx->drain_ev);
        if (ctx->drainer_stream) cudaStreamDestroy(ctx->drainer_stream);
    }
    delete ctx;
    return rc;
}

extern "C" int32_t cc_last_cuda_error(cc_ctx* ctx) { return ctx ? ctx->last_cuda : 0; }
#if CC_TRACE_ON
extern "C" int32_t cc_debug_trace(cc_ctx* ctx, uint64_t* out32) {       // probe builds only; not declared in concordia.h
    return cudaMemcpy(out32, ctx->d_dev->trace, sizeof(ctx->d_dev->trace), cudaMemcpyDeviceToHost) == cudaSuccess ? CC_OK : CC_ERR_CUDA;
}
#endif
extern "C" uint64_t cc_kernel_launches(cc_ctx* ctx) { return ctx ? ctx->launches : 0; }

// -------------------------------------------------------------------------- regions --

extern "C" uint64_t cc_workspace_bytes(uint64_t bytes, uint32_t page_bytes) {
    cc_ws_layout L;
    return ws_layout(bytes, page_bytes, &L) ? L.total : 0;
}

extern "C" int32_t cc_register_region(cc_ctx* ctx, const cc_region_desc* d) {
    if (!ctx || !d) return CC_ERR_INVALID;
    if (ctx->worker_running) return CC_ERR_WORKER;
    cc_ws_layout L;
    if (d->region_id == 0 || d->region_id == CC_COMMIT_ID || !ws_layout(d->bytes, d->page_bytes, &L)) return CC_ERR_INVALID;
    const bool no_shadow = (d->flags & CC_REG_NO_SHADOW) != 0;
    if (!d->base || !d->workspace || ((uintptr_t)d->base & 15) || ((uintptr_t)d->shadow & 15) ||
        ((uintptr_t)d->workspace & 255) || d->workspace_bytes < L.total)
        return CC_ERR_INVALID;
    if (no_shadow ? (d->shadow != nullptr || (d->flags & CC_REG_SNAPSHOT_NOW)) : (d->shadow == nullptr)) return CC_ERR_INVALID;
    if (find_slot(ctx, d->region_id) >= 0) return CC_ERR_EXISTS;
    int slot = -1;
    for (int s = 0; s < CC_MAX_REGIONS; s++)
        if (!ctx->regions[s].used) { slot = s; break; }
    if (slot < 0) return CC_ERR_INVALID;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    // Legacy default stream: ordered after whatever the caller queued on blocking streams.
    CC_CUDA(ctx, cudaMemsetAsync(d->workspace, 0, L.total, 0));
    if (d->flags & CC_REG_SNAPSHOT_NOW) CC_CUDA(ctx, cudaMemcpyAsync(d->shadow, d->base, d->bytes, cudaMemcpyDeviceToDevice, 0));
    cc_region_dev r;
    memset(&r, 0, sizeof(r));
    u8* ws = (u8*)d->workspace;
    r.base = (u8*)d->base;
    r.shadow = (u8*)d->shadow;
    r.bytes = d->bytes;
    r.n_pages = L.n_pages;
    r.page_bytes = d->page_bytes;
    r.region_id = d->region_id;
    r.spp = (d->page_bytes + CC_SEG_BYTES - 1) / CC_SEG_BYTES;
    r.spp_shift = -1;
    if ((r.spp & (r.spp - 1)) == 0) { r.spp_shift = 0; while ((1u << r.spp_shift) < r.spp) r.spp_shift++; }
    r.n_words = L.n_words;
    r.hdr = (cc_ws_hdr*)(ws + L.hdr);
    r.bitmap = (u32*)(ws + L.bitmap);
    r.D = (u32*)(ws + L.D);
    r.rec_state = (u64*)(ws + L.rec_state);
    r.latest = (u32*)(ws + L.latest);
    r.lb_status = (u64*)(ws + L.lb);
    r.flb_status = (u64*)(ws + L.flb);
    r.S = (u32*)(ws + L.S);
    r.Rfirst = (u32*)(ws + L.Rfirst);
    r.Rn = (u32*)(ws + L.Rn);
    r.run_state = (u64*)(ws + L.run_state);
    r.hdr2 = (cc_ws_hdr*)(ws + L.hdr2);
    r.lb2 = (u64*)(ws + L.lb2);
    r.ftile_pages = (u32)L.ftile_pages;
    r.n_ftiles = (u32)L.n_ftiles;
    {
        cc_crc_tables* t = (cc_crc_tables*)malloc(sizeof(cc_crc_tables));
        cc_crc_build_tables(t);
        const u64 tail = d->bytes - (L.n_pages - 1) * (u64)d->page_bytes;
        r.crc_init_full = gf_mul(0xFFFFFFFFu, gf_xpow_bytes(t->xp, d->page_bytes));
        r.crc_init_tail = gf_mul(0xFFFFFFFFu, gf_xpow_bytes(t->xp, tail));
        free(t);
    }
    const u32 one = 1;
    CC_CUDA(ctx, cudaMemcpyAsync(&ctx->d_dev->regions[slot], &r, sizeof(r), cudaMemcpyHostToDevice, 0));
    CC_CUDA(ctx, cudaMemcpyAsync(&ctx->d_dev->region_used[slot], &one, sizeof(one), cudaMemcpyHostToDevice, 0));
    CC_CUDA(ctx, cudaStreamSynchronize(0));
    ctx->regions[slot].used = true;
    ctx->regions[slot].desc = *d;
    ctx->regions[slot].dev = r;
    return CC_OK;
}

extern "C" int32_t cc_unregister_region(cc_ctx* ctx, uint32_t region_id) {
    if (!ctx) return CC_ERR_INVALID;
    if (ctx->worker_running) return CC_ERR_WORKER;
    int slot = find_slot(ctx, region_id);
    if (slot < 0) return CC_ERR_NOT_REGISTERED;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    const u32 zero = 0;
    CC_CUDA(ctx, cudaMemcpyAsync(&ctx->d_dev->region_used[slot], &zero, sizeof(zero), cudaMemcpyHostToDevice, 0));
    CC_CUDA(ctx, cudaStreamSynchronize(0));
    ctx->regions[slot].used = false;
    return CC_OK;
}

// ------------------------------------------------------------------------------ log --

extern "C" int32_t cc_log_attach(cc_ctx* ctx, void* log_buf, uint64_t capacity, uint64_t* committed_off) {
    if (!ctx || !log_buf || ((uintptr_t)log_buf & 15) || capacity < CC_COMMIT_RECORD_BYTES) return CC_ERR_INVALID;
    if (ctx->worker_running) return CC_ERR_WORKER;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cc_log_dev l;
    l.buf = (u8*)log_buf;
    l.capacity = capacity;
    l.W = 0;
    l.committed_off = committed_off;
    l.gen = 0;
    l.pub = (u64*)(ctx->ring_words + 24);
    if (ctx->drainer) return CC_ERR_INVALID;             // stop the drainer before re-attaching
    __atomic_store_n(ctx->ring_words + 24, 0ull, __ATOMIC_RELEASE);
    CC_CUDA(ctx, cudaMemcpyAsync(&ctx->d_dev->log, &l, sizeof(l), cudaMemcpyHostToDevice, 0));
    CC_CUDA(ctx, cudaStreamSynchronize(0));
    ctx->log_attached = true;
    ctx->committed_off = committed_off;
    {
        cudaPointerAttributes at;
        ctx->log_is_host = cudaPointerGetAttributes(&at, log_buf) == cudaSuccess && at.type == cudaMemoryTypeHost;
        cudaGetLastError();
    }
    ctx->log_buf = log_buf;
    ctx->log_capacity = capacity;
    ctx->drained = 0;
    return CC_OK;
}

__global__ void cc_log_reset_kernel(cc_dev* dev) { cc_log_rewind(&dev->log); }

extern "C" int32_t cc_log_reset(cc_ctx* ctx) {
    if (!ctx || !ctx->log_attached) return CC_ERR_INVALID;
    if (ctx->worker_running) return CC_ERR_WORKER;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cc_log_reset_kernel<<<1, 1, 0, 0>>>(ctx->d_dev);     // W := 0, next generation, publish the rewind too
    ctx->launches += 1;
    CC_CUDA(ctx, cudaGetLastError());
    CC_CUDA(ctx, cudaStreamSynchronize(0));
    if (!ctx->drainer) {                                 // (a running drainer thread follows the generation itself)
        ctx->drained = 0;
        if (ctx->mirror_committed) __atomic_store_n(ctx->mirror_committed, 0ull, __ATOMIC_RELEASE);
    }
    return CC_OK;
}

// ---- host mirror of a device-resident log, drained by the copy engine ----

struct cc_drain_note { uint64_t* word; uint64_t value; };
static void CUDART_CB cc_drain_publish(void* p) {
    cc_drain_note* nt = (cc_drain_note*)p;
    __atomic_store_n(nt->word, nt->value, __ATOMIC_RELEASE);     // after the bytes: stream order + release
    free(nt);
}

extern "C" int32_t cc_log_mirror_attach(cc_ctx* ctx, void* host_log, uint64_t capacity, uint64_t* committed_off_host) {
    if (!ctx || ((uintptr_t)host_log & 15) || ctx->drainer) return CC_ERR_INVALID;
    if (ctx->worker_running) return CC_ERR_WORKER;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    if (host_log && !ctx->drain_ev) CC_CUDA(ctx, cudaEventCreateWithFlags(&ctx->drain_ev, cudaEventDisableTiming));
    ctx->mirror = host_log;
    ctx->mirror_capacity = host_log ? capacity : 0;
    ctx->mirror_committed = host_log ? committed_off_host : nullptr;
    ctx->drained = 0;
    if (ctx->mirror_committed) __atomic_store_n(ctx->mirror_committed, 0ull, __ATOMIC_RELEASE);
    return CC_OK;
}

extern "C" int32_t cc_log_drain(cc_ctx* ctx, uint64_t upto, void* after_stream, void* copy_stream) {
    if (!ctx || !ctx->log_attached || !ctx->mirror || ctx->drainer) return CC_ERR_INVALID;
    if (upto < ctx->drained || upto > ctx->log_capacity) return CC_ERR_INVALID;
    if (upto > ctx->mirror_capacity) return CC_ERR_LOG_FULL;
    if (upto == ctx->drained) return CC_OK;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t cs = (cudaStream_t)copy_stream;
    CC_CUDA(ctx, cudaEventRecord(ctx->drain_ev, (cudaStream_t)after_stream));
    CC_CUDA(ctx, cudaStreamWaitEvent(cs, ctx->drain_ev, 0));
    // In pieces: a copy engine serves its queue one command at a time, and another stream's small copy that lands on the
    // same engine (the application's own H2D / D2H traffic) would otherwise wait behind the whole drain.
    const uint64_t piece = 16ull << 20;
    for (uint64_t o = ctx->drained; o < upto; o += piece) {
        const uint64_t nb = upto - o < piece ? upto - o : piece;
        CC_CUDA(ctx, cudaMemcpyAsync((u8*)ctx->mirror + o, (const u8*)ctx->log_buf + o, nb, cudaMemcpyDefault, cs));
    }
    if (ctx->mirror_committed) {
        cc_drain_note* nt = (cc_drain_note*)malloc(sizeof(cc_drain_note));
        if (!nt) return CC_ERR_INVALID;
        nt->word = ctx->mirror_committed;
        nt->value = upto;
        const cudaError_t e = cudaLaunchHostFunc(cs, cc_drain_publish, nt);
        if (e != cudaSuccess) { free(nt); ctx->last_cuda = (int)e; return CC_ERR_CUDA; }
    }
    ctx->drained = upto;
    return CC_OK;
}

extern "C" int32_t cc_log_reset_async(cc_ctx* ctx, void* stream) {
    if (!ctx || !ctx->log_attached) return CC_ERR_INVALID;
    if (ctx->worker_running) return CC_ERR_WORKER;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cc_log_reset_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(ctx->d_dev);
    ctx->launches += 1;
    CC_CUDA(ctx, cudaGetLastError());
    // the mirror's drain position and published offset rewind with the log: drains issued after this call (in host
    // order) copy from offset 0 again; the mirror's word is zeroed in stream order, like committed_off
    if (ctx->drainer) return CC_OK;                      // the drainer thread follows the generation by itself
    ctx->drained = 0;
    if (ctx->mirror_committed) {
        cc_drain_note* nt = (cc_drain_note*)malloc(sizeof(cc_drain_note));
        if (!nt) return CC_ERR_INVALID;
        nt->word = ctx->mirror_committed;
        nt->value = 0;
        const cudaError_t e = cudaLaunchHostFunc((cudaStream_t)stream, cc_drain_publish, nt);
        if (e != cudaSuccess) { free(nt); ctx->last_cuda = (int)e; return CC_ERR_CUDA; }
    }
    return CC_OK;
}

// ---- library-side drainer: staging buffer -> host log without a per-step call ----
// A host thread follows the library's published word (generation << 48 | committed offset, release-stored by the
// commit of every checkpoint, host-launched or worker) and hands every newly committed byte range of the
// device-resident log to the copy engine; after a range has landed it publishes the mirror's offset.  A log reset
// starts a new generation: the thread starts again at offset 0 of the mirror.

struct cc_landed_note { cc_ctx* ctx; uint64_t gen, upto; };
static void CUDART_CB cc_drain_landed(void* p) {
    cc_landed_note* nt = (cc_landed_note*)p;
    cc_ctx* c = nt->ctx;
    if (c->drainer_gen.load(std::memory_order_acquire) == nt->gen) {
        if (c->mirror_committed) __atomic_store_n(c->mirror_committed, nt->upto, __ATOMIC_RELEASE);
        c->drainer_landed.store(nt->upto, std::memory_order_release);
    }
    free(nt);
}

static void cc_drainer_main(cc_ctx* ctx) {
    if (cudaSetDevice(ctx->device) != cudaSuccess) { ctx->drainer_status.store(CC_ERR_CUDA); return; }
    cudaStream_t cs = ctx->drainer_stream;
    uint64_t gen = ctx->drainer_gen.load(), drained = ctx->drainer_landed.load();
    const uint64_t piece = 16ull << 20;
    uint32_t idle = 0;
    for (;;) {
        const bool stopping = ctx->drainer_stop.load(std::memory_order_acquire) != 0;
        const uint64_t pub = __atomic_load_n(ctx->ring_words + 24, __ATOMIC_ACQUIRE);
        const uint64_t g = pub >> CC_PUB_SHIFT, c = pub & ((1ull << CC_PUB_SHIFT) - 1);
        if (g != gen) {                                  // the log was reset: a new generation starts at offset 0
            cudaStreamSynchronize(cs);                   // copies of the old generation finish first
            gen = g;
            drained = 0;
            ctx->drainer_landed.store(0, std::memory_order_release);
            ctx->drainer_gen.store(g, std::memory_order_release);
            if (ctx->mirror_committed) __atomic_store_n(ctx->mirror_committed, 0ull, __ATOMIC_RELEASE);
        }
        if (c > drained) {
            idle = 0;
            if (c > ctx->mirror_capacity) { ctx->drainer_status.store(CC_ERR_LOG_FULL); return; }
            cudaError_t e = cudaSuccess;
            for (uint64_t o = drained; o < c && e == cudaSuccess; o += piece) {
                const uint64_t nb = c - o < piece ? c - o : piece;
                e = cudaMemcpyAsync((u8*)ctx->mirror + o, (const u8*)ctx->log_buf + o, nb, cudaMemcpyDefault, cs);
            }
            cc_landed_note* nt = (cc_landed_note*)malloc(sizeof(cc_landed_note));
            if (e == cudaSuccess && nt) {
                nt->ctx = ctx; nt->gen = gen; nt->upto = c;
                e = cudaLaunchHostFunc(cs, cc_drain_landed, nt);
                if (e != cudaSuccess) free(nt);
            } else if (nt) free(nt);
            if (e != cudaSuccess || !nt) { ctx->last_cuda = (int)e; ctx->drainer_status.store(CC_ERR_CUDA); return; }
            drained = c;
            continue;
        }
        if (stopping) break;
        if (++idle < 2000) {
#if defined(__x86_64__)
            __builtin_ia32_pause();
#endif
        } else {
            struct timespec ts = {0, 20000};             // 20 us naps once nothing has been committed for a while
            nanosleep(&ts, nullptr);
        }
    }
    cudaStreamSynchronize(cs);
}

extern "C" int32_t cc_log_drain_start(cc_ctx* ctx) {
    if (!ctx || !ctx->log_attached || !ctx->mirror) return CC_ERR_INVALID;
    if (ctx->drainer) return CC_ERR_EXISTS;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    if (!ctx->drainer_stream) CC_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->drainer_stream, cudaStreamNonBlocking));
    const uint64_t pub = __atomic_load_n(ctx->ring_words + 24, __ATOMIC_ACQUIRE);
    ctx->drainer_gen.store(pub >> CC_PUB_SHIFT);
    ctx->drainer_landed.store(ctx->drained);             // what cc_log_drain has already carried over
    ctx->drainer_stop.store(0);
    ctx->drainer_status.store(CC_OK);
    ctx->drainer = new (std::nothrow) std::thread(cc_drainer_main, ctx);
    return ctx->drainer ? CC_OK : CC_ERR_INVALID;
}

extern "C" int32_t cc_log_drain_wait(cc_ctx* ctx, uint64_t upto, uint64_t timeout_ns) {
    if (!ctx || !ctx->drainer) return CC_ERR_INVALID;
    const auto t0 = std::chrono::steady_clock::now();
    for (;;) {
        // "landed" counts bytes of the generation the thread is on: it must be the log's current one
        const uint64_t g = __atomic_load_n(ctx->ring_words + 24, __ATOMIC_ACQUIRE) >> CC_PUB_SHIFT;
        if (ctx->drainer_gen.load(std::memory_order_acquire) == g && ctx->drainer_landed.load(std::memory_order_acquire) >= upto) return CC_OK;
        const int32_t st = ctx->drainer_status.load();
        if (st != CC_OK) return st;
        if ((uint64_t)std::chrono::duration_cast<std::chrono::nanoseconds>(std::chrono::steady_clock::now() - t0).count() > timeout_ns)
            return CC_ERR_TIMEOUT;
#if defined(__x86_64__)
        __builtin_ia32_pause();
#endif
    }
}

extern "C" int32_t cc_log_drain_stop(cc_ctx* ctx) {
    if (!ctx || !ctx->drainer) return CC_ERR_INVALID;
    ctx->drainer_stop.store(1, std::memory_order_release);
    ctx->drainer->join();
    delete ctx->drainer;
    ctx->drainer = nullptr;
    ctx->drained = ctx->drainer_landed.load();
    return ctx->drainer_status.load();
}

// ------------------------------------------------------------- host-launched path --

// Launch `kernel` so that it may begin while the previous kernel of the stream is still running (programmatic dependent
// launch); the kernel waits with cc_pdl_wait() before it reads that kernel's results.
template <typename... KArgs, typename... Args>
static cudaError_t launch_dependent(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st, Args... args) {
#if CC_PDL
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
#else
    kernel<<<grid, block, smem, st>>>(KArgs(args)...);
    return cudaGetLastError();
#endif
}

static int32_t launch_compact(cc_ctx* ctx, int slot, u32 mode, uint64_t epoch, cudaStream_t st, cc_result* out) {
    const cc_region_dev& r = ctx->regions[slot].dev;
    const uint64_t n_tiles = (r.n_words + CC_COMPACT_TILE_WORDS - 1) / CC_COMPACT_TILE_WORDS;
    uint64_t g2 = n_tiles < (uint64_t)ctx->sm_count * 4 ? n_tiles : (uint64_t)ctx->sm_count * 4;
    CC_CUDA(ctx, launch_dependent(cc_compact_kernel, (unsigned)g2, CC_COMPACT_THREADS, 0, st, ctx->d_dev, ctx->regions[slot].dev, mode, epoch, out));
    if (ctx->ev_after_compact) cudaEventRecord(ctx->ev_after_compact, st);
    ctx->launches += 1;
    return CC_OK;
}

static int32_t launch_scan_compact(cc_ctx* ctx, int slot, u32 mode, uint64_t epoch, cudaStream_t st, cc_result* out) {
    const cc_region_dev& r = ctx->regions[slot].dev;
    const uint64_t n_items = r.n_pages * (uint64_t)r.spp;
    const uint64_t wpb = CC_SCAN_THREADS / 32;
    uint64_t g1 = (n_items + wpb - 1) / wpb;
    const uint64_t cap1 = (uint64_t)ctx->sm_count * ctx->scan_bps;
    if (g1 > cap1) g1 = cap1;
    cc_scan_kernel<<<(unsigned)g1, CC_SCAN_THREADS, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev);
    if (ctx->ev_after_scan) cudaEventRecord(ctx->ev_after_scan, st);
    ctx->launches += 1;
    return launch_compact(ctx, slot, mode, epoch, st, out);
}

static int32_t launch_gather(cc_ctx* ctx, int slot, cudaStream_t st, cc_result* out) {
    const unsigned g3 = (unsigned)(ctx->sm_count * ctx->gather_bps);
    CC_CUDA(ctx, launch_dependent(cc_gather_kernel, g3, CC_GATHER_THREADS, sizeof(cc_crc_smem), st, ctx->d_dev, ctx->regions[slot].dev, out));
    ctx->launches += 1;
    return CC_OK;
}

static unsigned small_grid(cc_ctx* ctx, uint64_t items, uint64_t per_block) {
    uint64_t g = (items + per_block - 1) / per_block;
    const uint64_t cap = (uint64_t)ctx->sm_count * 8;
    if (g > cap) g = cap;
    return (unsigned)(g < 1 ? 1 : g);
}

// ---- one checkpoint of one region: the general entry point and its path selection ----
#ifndef CC_PASS_COOP
#define CC_PASS_COOP 1              // 0: plain launch (A/B of the launch cost only: the kernel NEEDS co-residency)
#endif

// Single pass (ONE cooperative launch).
static int32_t launch_pass(cc_ctx* ctx, int slot, const cc_pass_args& a, cudaStream_t st, cc_result* out) {
    const cc_region_dev& r = ctx->regions[slot].dev;
    uint64_t g = (r.n_pages + CC_GATHER_THREADS / 32 - 1) / (CC_GATHER_THREADS / 32);
    const uint64_t cap = (uint64_t)ctx->sm_count * ctx->fused_bps;       // all blocks co-resident (grid barrier of the fallback)
    if (g > cap) g = cap;
    cc_dev* d = ctx->d_dev;
    cc_pass_args aa = a;
    cc_region_dev rgv = ctx->regions[slot].dev;
    void* args[] = {&d, &rgv, &aa, &out};
#if CC_PASS_COOP
    CC_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)cc_pass_kernel, dim3((unsigned)g), dim3(CC_GATHER_THREADS), args,
                                             sizeof(cc_crc_smem), st));
#else
    (void)args;
    cc_pass_kernel<<<(unsigned)g, CC_GATHER_THREADS, sizeof(cc_crc_smem), st>>>(d, rgv, aa, out);
    CC_CUDA(ctx, cudaGetLastError());
#endif
    ctx->launches += 1;
    if (ctx->ev_after_scan) cudaEventRecord(ctx->ev_after_scan, st);
    if (ctx->ev_after_compact) cudaEventRecord(ctx->ev_after_compact, st);
    return CC_OK;
}

// Small-region path (ONE cooperative launch, cc_small.cuh): as many blocks as the scan has work for, all co-resident.
static int32_t launch_small(cc_ctx* ctx, int slot, uint64_t epoch, cudaStream_t st, cc_result* out) {
    const cc_region_dev& r = ctx->regions[slot].dev;
    const uint64_t n_items = r.n_pages * (uint64_t)r.spp;
    uint64_t g = (n_items + CC_GATHER_THREADS / 32 - 1) / (CC_GATHER_THREADS / 32);
    const uint64_t cap = (uint64_t)ctx->sm_count * ctx->small_bps;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    cc_dev* d = ctx->d_dev;
    cc_region_dev rgv = ctx->regions[slot].dev;
    void* args[] = {&d, &rgv, &epoch, &out};
    CC_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)cc_small_kernel, dim3((unsigned)g), dim3(CC_GATHER_THREADS), args,
                                             sizeof(cc_crc_smem), st));
    ctx->launches += 1;
    if (ctx->ev_after_scan) cudaEventRecord(ctx->ev_after_scan, st);
    if (ctx->ev_after_compact) cudaEventRecord(ctx->ev_after_compact, st);
    return CC_OK;
}

// Classic phases as separate launches, each sized for its own work (the scanner runs at 47 warps per SM).
static int32_t launch_phases(cc_ctx* ctx, int slot, const cc_pass_args& a, cudaStream_t st, cc_result* out) {
    const cc_region_dev& r = ctx->regions[slot].dev;
    const bool rle = a.run_pages > 1;
    const u32 final_mode = rle ? CC_MODE_SCAN_ONLY : CC_MODE_CHECKPOINT;
    cudaEvent_t ec = ctx->ev_after_compact;
    int32_t rc = CC_OK;
    if (a.disc == CC_DISC_SCAN && !rle && cc_small_supported(r.n_words) && r.bytes <= CC_SMALL_TAIL_MAX_BYTES) {
        // latency-bound sizes: the scan kernel, then ONE kernel in which every block ranks the bitmap by itself and the
        // records follow at once (cc_small.cuh) -- the compaction kernel and its launch gap are 8 us of a 50 us call
        const uint64_t n_items = r.n_pages * (uint64_t)r.spp;
        uint64_t g1 = (n_items + CC_SCAN_THREADS / 32 - 1) / (CC_SCAN_THREADS / 32);
        const uint64_t cap1 = (uint64_t)ctx->sm_count * ctx->scan_bps;
        if (g1 > cap1) g1 = cap1;
        cc_scan_kernel<<<(unsigned)g1, CC_SCAN_THREADS, 0, st>>>(ctx->d_dev, r);
        if (ctx->ev_after_scan) cudaEventRecord(ctx->ev_after_scan, st);
        if (ec) cudaEventRecord(ec, st);
        uint64_t g2 = (n_items + CC_GATHER_THREADS / 32 - 1) / (CC_GATHER_THREADS / 32);
        const uint64_t cap2 = (uint64_t)ctx->sm_count * ctx->small_bps;
        if (g2 > cap2) g2 = cap2;
        if (g2 < 1) g2 = 1;
        cc_small_tail_kernel<<<(unsigned)g2, CC_GATHER_THREADS, sizeof(cc_crc_smem), st>>>(ctx->d_dev, r, a.epoch, out);
        ctx->launches += 2;
        CC_CUDA(ctx, cudaGetLastError());
        return CC_OK;
    }
    if (a.disc == CC_DISC_SCAN) {
        if (rle) ctx->ev_after_compact = nullptr;             // the trace event goes after the whole ranking
        rc = launch_scan_compact(ctx, slot, final_mode, a.epoch, st, nullptr);
        ctx->ev_after_compact = ec;
    } else if (a.disc == CC_DISC_ALL) {
        cc_snapshot_plan_kernel<<<small_grid(ctx, r.n_pages, 256), 256, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev, a.epoch);
        ctx->launches += 1;
        if (ctx->ev_after_scan) cudaEventRecord(ctx->ev_after_scan, st);
        if (ec && !rle) cudaEventRecord(ec, st);
    } else {
        if (a.disc == CC_DISC_VERSIONS)
            cc_mark_versions_kernel<<<small_grid(ctx, r.n_words, 8), 256, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev, a.version, a.committed);
        else
            cc_mark_load_kernel<<<small_grid(ctx, r.n_words, 256), 256, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev, a.marks);
        ctx->launches += 1;
        ctx->ev_after_compact = nullptr;                      // the trace events bracket discovery as a whole
        if (a.disc == CC_DISC_MARKS_VERIFY) {
            rc = launch_compact(ctx, slot, CC_MODE_SCAN_ONLY, a.epoch, st, nullptr);
            if (rc == CC_OK) {
                cc_mark_verify_kernel<<<(unsigned)(ctx->sm_count * ctx->scan_bps), CC_SCAN_THREADS, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev);
                ctx->launches += 1;
            }
        }
        if (ctx->ev_after_scan) cudaEventRecord(ctx->ev_after_scan, st);
        if (!rle) ctx->ev_after_compact = ec;
        if (rc == CC_OK) rc = launch_compact(ctx, slot, final_mode, a.epoch, st, nullptr);
        ctx->ev_after_compact = ec;
    }
    if (rc != CC_OK) return rc;
    if (rle) {
        const uint64_t n_tiles = (r.n_words + CC_COMPACT_TILE_WORDS - 1) / CC_COMPACT_TILE_WORDS;
        const unsigned g2 = (unsigned)(n_tiles < (uint64_t)ctx->sm_count * 4 ? n_tiles : (uint64_t)ctx->sm_count * 4);
        cc_rle_starts_kernel<<<small_grid(ctx, r.n_words, 8), 256, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev, a.run_pages);
        cc_rle_rank_kernel<<<g2, CC_COMPACT_THREADS, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev);
        cc_rle_plan_kernel<<<small_grid(ctx, r.n_pages, 256), 256, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev, a.epoch);
        if (ec) cudaEventRecord(ec, st);
        cc_rle_gather_kernel<<<(unsigned)(ctx->sm_count * ctx->gather_bps), CC_GATHER_THREADS, sizeof(cc_crc_smem), st>>>(ctx->d_dev, ctx->regions[slot].dev, out);
        ctx->launches += 4;
        CC_CUDA(ctx, cudaGetLastError());
    } else {
        rc = launch_gather(ctx, slot, st, out);
        if (rc != CC_OK) return rc;
    }
    if ((a.disc == CC_DISC_MARKS || a.disc == CC_DISC_MARKS_VERIFY) && a.consume) {
        cc_mark_finish_kernel<<<small_grid(ctx, r.n_words, 256), 256, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev, a.marks, nullptr, nullptr);
        ctx->launches += 1;
    } else if (a.disc == CC_DISC_VERSIONS) {
        cc_mark_finish_kernel<<<small_grid(ctx, r.n_pages, 256), 256, 0, st>>>(ctx->d_dev, ctx->regions[slot].dev, nullptr, a.version, a.committed);
        ctx->launches += 1;
    }
    CC_CUDA(ctx, cudaGetLastError());
    return CC_OK;
}

extern "C" int32_t cc_checkpoint_ex(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, const cc_ckpt_opts* o, void* stream, cc_result* out) {
    if (!ctx) return CC_ERR_INVALID;
    CC_NO_WORKER(ctx);
    cc_ckpt_opts z;
    memset(&z, 0, sizeof(z));
    if (o) z = *o;
    if (z.discovery > CC_DISC_ALL || z.path > CC_PATH_SMALL || (z.mark_flags & ~(CC_MARK_VERIFY | CC_MARK_CONSUME))) return CC_ERR_INVALID;
    int slot = find_slot(ctx, region_id);
    if (slot < 0) return CC_ERR_NOT_REGISTERED;
    const cc_region_dev& r = ctx->regions[slot].dev;
    cc_pass_args a;
    memset(&a, 0, sizeof(a));
    a.epoch = epoch;
    a.run_pages = z.run_pages;
    a.kind = CC_TASK_DELTA_CKPT;
    if (z.run_pages > 1 && (uint64_t)z.run_pages * r.page_bytes > 0xFFFFFFFFull) return CC_ERR_INVALID;
    switch (z.discovery) {
    case CC_DISC_SCAN:
        if (!r.shadow) return CC_ERR_INVALID;
        a.disc = CC_DISC_SCAN;
        break;
    case CC_DISC_MARKS:
        if (!z.dirty_bitmap || ((uintptr_t)z.dirty_bitmap & 3)) return CC_ERR_INVALID;
        if ((z.mark_flags & CC_MARK_VERIFY) && !r.shadow) return CC_ERR_INVALID;
        a.disc = (z.mark_flags & CC_MARK_VERIFY) ? CC_DISC_MARKS_VERIFY : CC_DISC_MARKS;
        a.marks = z.dirty_bitmap;
        a.consume = (z.mark_flags & CC_MARK_CONSUME) ? 1u : 0u;
        a.kind = CC_TASK_MARKED_CKPT;
        break;
    case CC_DISC_VERSIONS:
        if (!z.version || !z.committed || ((uintptr_t)z.version & 7) || ((uintptr_t)z.committed & 7)) return CC_ERR_INVALID;
        a.disc = CC_DISC_VERSIONS;
        a.version = z.version;
        a.committed = z.committed;
        a.kind = CC_TASK_VERSION_CKPT;
        break;
    default:
        a.disc = CC_DISC_ALL;
        a.kind = CC_TASK_SNAPSHOT;
        break;
    }
    if (z.discovery == CC_DISC_MARKS_VERIFY) return CC_ERR_INVALID;      // (spelled CC_DISC_MARKS + CC_MARK_VERIFY)
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    const bool can_pass = cc_pass_supported(r.n_pages, z.run_pages);
    const bool can_small = a.disc == CC_DISC_SCAN && z.run_pages <= 1 && cc_small_supported(r.n_words);
    if (z.path == CC_PATH_SMALL) {
        if (!can_small) return CC_ERR_INVALID;
        return launch_small(ctx, slot, epoch, (cudaStream_t)stream, out);
    }
    bool pass;
    if (z.path == CC_PATH_SINGLE_PASS) {
        if (!can_pass) return CC_ERR_INVALID;
        pass = true;
    } else if (z.path == CC_PATH_PHASES) pass = false;
    else {
        // AUTO, from measurements (profiles/r02_small_region.md, profiles/r02_pass_probe.md): with a
        // device log the separately sized kernels win at every size (64 MiB: 46 us as scan + tail kernel against 55 us for
        // the one-launch small path and 62 us for the single pass; 8 GiB: 2.75 vs 3.2 ms); the single pass wins where the records cross the host link while it scans (8 GiB: 12.0 vs 13.8 ms,
        // 256 MiB ring task: 110 vs 150 us) -- but not on regions so small that its per-tile ranking costs more than the
        // transfer (64 MiB: 66 vs 56 us).
        pass = can_pass && ctx->log_is_host && r.bytes >= CC_PASS_AUTO_MIN_BYTES;
    }
    return pass ? launch_pass(ctx, slot, a, (cudaStream_t)stream, out) : launch_phases(ctx, slot, a, (cudaStream_t)stream, out);
}

static int32_t checkpoint_opts(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, void* stream, cc_result* out, uint32_t disc,
                               uint32_t path, uint32_t run_pages, uint32_t* marks, uint32_t mark_flags, const uint64_t* version,
                               uint64_t* committed) {
    cc_ckpt_opts o;
    memset(&o, 0, sizeof(o));
    o.discovery = disc; o.path = path; o.run_pages = run_pages; o.dirty_bitmap = marks; o.mark_flags = mark_flags;
    o.version = version; o.committed = committed;
    return cc_checkpoint_ex(ctx, region_id, epoch, &o, stream, out);
}

extern "C" int32_t cc_checkpoint_delta(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, void* stream, cc_result* out) {
    return checkpoint_opts(ctx, region_id, epoch, stream, out, CC_DISC_SCAN, CC_PATH_AUTO, 0, nullptr, 0, nullptr, nullptr);
}

extern "C" int32_t cc_checkpoint_delta_fused(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, void* stream, cc_result* out) {
    return checkpoint_opts(ctx, region_id, epoch, stream, out, CC_DISC_SCAN, CC_PATH_SINGLE_PASS, 0, nullptr, 0, nullptr, nullptr);
}

extern "C" int32_t cc_checkpoint_delta_rle(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, uint32_t run_pages, void* stream,
                                           cc_result* out) {
    if (run_pages == 0) return CC_ERR_INVALID;
    return checkpoint_opts(ctx, region_id, epoch, stream, out, CC_DISC_SCAN, run_pages <= 32 ? CC_PATH_AUTO : CC_PATH_PHASES, run_pages,
                           nullptr, 0, nullptr, nullptr);
}

extern "C" int32_t cc_checkpoint_marked(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, uint32_t* dirty_bitmap,
                                        uint32_t flags, void* stream, cc_result* out) {
    if (!dirty_bitmap) return CC_ERR_INVALID;
    return checkpoint_opts(ctx, region_id, epoch, stream, out, CC_DISC_MARKS, CC_PATH_AUTO, 0, dirty_bitmap, flags, nullptr, nullptr);
}

extern "C" int32_t cc_checkpoint_versions(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, const uint64_t* version,
                                          uint64_t* committed, void* stream, cc_result* out) {
    if (!version || !committed) return CC_ERR_INVALID;
    return checkpoint_opts(ctx, region_id, epoch, stream, out, CC_DISC_VERSIONS, CC_PATH_AUTO, 0, nullptr, 0, version, committed);
}

extern "C" int32_t cc_snapshot_region(cc_ctx* ctx, uint32_t region_id, uint64_t epoch, void* stream, cc_result* out) {
    return checkpoint_opts(ctx, region_id, epoch, stream, out, CC_DISC_ALL, CC_PATH_AUTO, 0, nullptr, 0, nullptr, nullptr);
}

extern "C" int32_t cc_checkpoint_all(cc_ctx* ctx, uint64_t epoch, void* stream, cc_result* out) {
    if (!ctx) return CC_ERR_INVALID;
    CC_NO_WORKER(ctx);
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    cc_batch_scan_kernel<<<(unsigned)(ctx->sm_count * ctx->scan_bps), CC_SCAN_THREADS, 0, st>>>(ctx->d_dev);
    if (ctx->ev_after_scan) cudaEventRecord(ctx->ev_after_scan, st);
    cc_batch_rank_kernel<<<(unsigned)ctx->sm_count, CC_COMPACT_THREADS, 0, st>>>(ctx->d_dev, epoch);
    cc_batch_plan_kernel<<<1, CC_MAX_REGIONS, 0, st>>>(ctx->d_dev, epoch);
    if (ctx->ev_after_compact) cudaEventRecord(ctx->ev_after_compact, st);
    cc_batch_gather_kernel<<<(unsigned)(ctx->sm_count * ctx->gather_bps), CC_GATHER_THREADS, sizeof(cc_crc_smem), st>>>(ctx->d_dev, out);
    ctx->launches += 4;
    CC_CUDA(ctx, cudaGetLastError());
    return CC_OK;
}

extern "C" int32_t cc_checkpoint_all_rle(cc_ctx* ctx, uint64_t epoch, uint32_t run_pages, void* stream, cc_result* out) {
    if (!ctx || run_pages == 0) return CC_ERR_INVALID;
    CC_NO_WORKER(ctx);
    // the regions that take part, in ascending region_id order
    cc_slot_list L;
    L.n = 0;
    for (int s = 0; s < CC_MAX_REGIONS; s++) {
        if (!ctx->regions[s].used || !ctx->regions[s].dev.shadow) continue;
        if ((uint64_t)run_pages * ctx->regions[s].dev.page_bytes > 0xFFFFFFFFull) return CC_ERR_INVALID;
        int i = L.n++;
        while (i > 0 && ctx->regions[L.slot[i - 1]].dev.region_id > ctx->regions[s].dev.region_id) { L.slot[i] = L.slot[i - 1]; i--; }
        L.slot[i] = s;
    }
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    cc_pass_args a;
    memset(&a, 0, sizeof(a));
    a.epoch = epoch;
    a.disc = CC_DISC_SCAN;
    a.run_pages = run_pages;
    a.kind = CC_TASK_DELTA_CKPT;
    for (int i = 0; i < L.n; i++) {
        const cc_region_dev& r = ctx->regions[L.slot[i]].dev;
        const int32_t rc = cc_pass_supported(r.n_pages, run_pages) ? launch_pass(ctx, L.slot[i], a, st, nullptr)
                                                                   : launch_phases(ctx, L.slot[i], a, st, nullptr);
        if (rc != CC_OK) return rc;
    }
    cc_batch_collect_kernel<<<1, 1, 0, st>>>(ctx->d_dev, L, epoch, 0ull, out);
    ctx->launches += 1;
    CC_CUDA(ctx, cudaGetLastError());
    return CC_OK;
}

// the four parse launches (candidates, their ordering, walks, serial fallback)
static void launch_parse(cc_ctx* ctx, const u8* lg, uint64_t nbytes, cudaStream_t st) {
    const uint64_t chunks = ((nbytes >> 4) + 255) >> 8;                              // 4 KiB per warp and step
    uint64_t gc = (chunks + CC_CAND_THREADS / 32 - 1) / (CC_CAND_THREADS / 32);
    const uint64_t capc = (uint64_t)ctx->sm_count * ctx->cand_bps;
    if (gc > capc) gc = capc;
    if (gc < 1) gc = 1;
    cc_apply_cand_kernel<<<(unsigned)gc, CC_CAND_THREADS, 0, st>>>(ctx->d_dev, ctx->tabs, lg, nbytes);
    launch_dependent(cc_apply_sort_kernel, (unsigned)ctx->sm_count, CC_SORT_THREADS, 0, st, ctx->d_dev, ctx->tabs);
    launch_dependent(cc_apply_walk_kernel, (unsigned)(ctx->sm_count * 4), CC_WALK_THREADS, 0, st, ctx->d_dev, ctx->tabs, lg, nbytes);
    launch_dependent(cc_apply_parse_kernel, 1u, CC_PARSE_THREADS, 0, st, ctx->d_dev, ctx->tabs, lg, nbytes);
    ctx->launches += 4;
}

extern "C" int32_t cc_compact_log(cc_ctx* ctx, const void* in_log, uint64_t in_bytes, void* out_log, uint64_t out_capacity,
                                  void* stream, cc_result* out) {
    if (!ctx || !in_log || !out_log || ((uintptr_t)in_log & 15) || ((uintptr_t)out_log & 15)) return CC_ERR_INVALID;
    CC_NO_WORKER(ctx);
    if (!ctx->apply_attached) return CC_ERR_INVALID;
    const uintptr_t a0 = (uintptr_t)in_log, a1 = a0 + in_bytes, b0 = (uintptr_t)out_log, b1 = b0 + out_capacity;
    if (a0 < b1 && b0 < a1) return CC_ERR_INVALID;       // the two logs must not overlap
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const u8* lg = stage_log(ctx, in_log, in_bytes, st);
    const unsigned gv = (unsigned)(ctx->sm_count * ctx->validate_bps);
    launch_parse(ctx, lg, in_bytes, st);
    launch_dependent(cc_apply_validate_kernel, gv, CC_VALIDATE_THREADS, sizeof(cc_crc_smem4), st, ctx->d_dev, ctx->tabs, lg);
    cc_compactor_mark_kernel<<<(unsigned)ctx->sm_count, CC_APPLY_THREADS, 0, st>>>(ctx->d_dev, ctx->tabs);
    cc_compactor_rank_kernel<<<(unsigned)ctx->sm_count, CC_COMPACT_THREADS, 0, st>>>(ctx->d_dev);
    cc_compactor_plan_kernel<<<1, CC_MAX_REGIONS, 0, st>>>(ctx->d_dev, out_capacity);
    cc_compactor_copy_kernel<<<gv, CC_APPLY_THREADS, sizeof(cc_crc_smem), st>>>(ctx->d_dev, ctx->tabs, lg, (u8*)out_log);
    cc_compactor_cleanup_kernel<<<(unsigned)ctx->sm_count, CC_APPLY_THREADS, 0, st>>>(ctx->d_dev, ctx->tabs, out);
    ctx->launches += 6;
    CC_CUDA(ctx, cudaGetLastError());
    return CC_OK;
}

extern "C" int32_t cc_scan_only(cc_ctx* ctx, uint32_t region_id, void* stream, cc_result* out) {
    if (!ctx) return CC_ERR_INVALID;
    CC_NO_WORKER(ctx);
    int slot = find_slot(ctx, region_id);
    if (slot < 0) return CC_ERR_NOT_REGISTERED;
    if (!ctx->regions[slot].dev.shadow) return CC_ERR_INVALID;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_scan_compact(ctx, slot, CC_MODE_SCAN_ONLY, 0, (cudaStream_t)stream, out);
}

#if CC_BENCH_HOOKS
extern "C" int32_t cc_trace_events(cc_ctx* ctx, void* ev_after_scan, void* ev_after_compact) {
    if (!ctx) return CC_ERR_INVALID;
    ctx->ev_after_scan = (cudaEvent_t)ev_after_scan;
    ctx->ev_after_compact = (cudaEvent_t)ev_after_compact;
    return CC_OK;
}
#endif

extern "C" int32_t cc_dirty_list(cc_ctx* ctx, uint32_t region_id, const uint32_t** d_list, const uint32_t** d_count) {
    if (!ctx) return CC_ERR_INVALID;
    int slot = find_slot(ctx, region_id);
    if (slot < 0) return CC_ERR_NOT_REGISTERED;
    if (d_list) *d_list = ctx->regions[slot].dev.D;
    if (d_count) *d_count = &ctx->regions[slot].dev.hdr->k;
    return CC_OK;
}

extern "C" uint64_t cc_apply_scratch_bytes(uint64_t max_records) {
    if (max_records == 0 || max_records >= 0x7FFFFFF0ull) return 0;      // record numbers travel in 31 bits
    return align_up(max_records * sizeof(cc_rec), 256) + align_up((max_records + 1) * sizeof(cc_epoch_ent), 256) +
           align_up(max_records * 8, 256) + align_up((max_records + 1) * 4, 256) +
           2 * align_up((max_records + 1) * 4, 256) + align_up((max_records + 2) * 8, 256);
}

extern "C" int32_t cc_apply_attach(cc_ctx* ctx, void* scratch, uint64_t scratch_bytes) {
    if (!ctx || !scratch || ((uintptr_t)scratch & 255)) return CC_ERR_INVALID;
    if (ctx->worker_running) return CC_ERR_WORKER;
    // largest max_records whose tables fit
    uint64_t lo = 0, hi = scratch_bytes / 64 + 2;
    while (lo + 1 < hi) {
        uint64_t mid = (lo + hi) / 2;
        uint64_t need = cc_apply_scratch_bytes(mid);
        if (need != 0 && need <= scratch_bytes) lo = mid; else hi = mid;
    }
    if (lo == 0) return CC_ERR_INVALID;
    const uint64_t m = lo;
    u8* p = (u8*)scratch;
    cc_apply_tabs T;
    T.max_records = m;
    T.recs = (cc_rec*)p; p += align_up(m * sizeof(cc_rec), 256);
    T.epochs = (cc_epoch_ent*)p; p += align_up((m + 1) * sizeof(cc_epoch_ent), 256);
    T.rec_state = (u64*)p; p += align_up(m * 8, 256);
    T.seg_begin = (u32*)p; p += align_up((m + 1) * 4, 256);
    T.cand = (u32*)p; p += align_up((m + 1) * 4, 256);
    T.cand_raw = (u32*)p; p += align_up((m + 1) * 4, 256);
    T.span_status = (u64*)p;
    ctx->tabs = T;
    ctx->apply_attached = true;
    return CC_OK;
}

extern "C" int32_t cc_apply_stage_attach(cc_ctx* ctx, void* device_buf, uint64_t bytes) {
    if (!ctx || ((uintptr_t)device_buf & 15)) return CC_ERR_INVALID;
    if (ctx->worker_running) return CC_ERR_WORKER;
    ctx->stage = bytes ? device_buf : nullptr;
    ctx->stage_bytes = device_buf ? bytes : 0;
    return CC_OK;
}

// A host-resident log is read twice by the kernels (validate, then scatter / copy): with a staging buffer
// attached it crosses the host link once, by the copy engine, and the kernels read the device copy.
static const u8* stage_log(cc_ctx* ctx, const void* log, uint64_t nbytes, cudaStream_t st) {
    if (!ctx->stage || nbytes == 0) return (const u8*)log;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, log) != cudaSuccess) { cudaGetLastError(); return (const u8*)log; }
    if (at.type != cudaMemoryTypeHost) return (const u8*)log;
    // a host-resident log with a staging buffer attached: from here on every way out is counted (cc_apply_stage_stats),
    // because reading the log in place costs three passes over the host link instead of one
    if (nbytes > ctx->stage_bytes ||
        cudaMemcpyAsync(ctx->stage, log, nbytes, cudaMemcpyHostToDevice, st) != cudaSuccess) {
        cudaGetLastError();
        ctx->stage_bypassed += 1;
        return (const u8*)log;
    }
    ctx->stage_used += 1;
    return (const u8*)ctx->stage;
}

extern "C" int32_t cc_apply_stage_stats(cc_ctx* ctx, uint64_t* staged, uint64_t* bypassed) {
    if (!ctx) return CC_ERR_INVALID;
    if (staged) *staged = ctx->stage_used;
    if (bypassed) *bypassed = ctx->stage_bypassed;
    return CC_OK;
}

extern "C" int32_t cc_apply_log(cc_ctx* ctx, const void* log, uint64_t nbytes, void* stream, cc_result* out) {
    if (!ctx || !log || ((uintptr_t)log & 15)) return CC_ERR_INVALID;
    CC_NO_WORKER(ctx);
    if (!ctx->apply_attached) return CC_ERR_INVALID;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const u8* lg = stage_log(ctx, log, nbytes, st);
    const unsigned gv = (unsigned)(ctx->sm_count * ctx->validate_bps);
    const unsigned gs = (unsigned)(ctx->sm_count * 8);
    launch_parse(ctx, lg, nbytes, st);
    launch_dependent(cc_apply_validate_kernel, gv, CC_VALIDATE_THREADS, sizeof(cc_crc_smem4), st, ctx->d_dev, ctx->tabs, lg);
    launch_dependent(cc_apply_latest_kernel, (unsigned)ctx->sm_count, CC_APPLY_THREADS, 0, st, ctx->d_dev, ctx->tabs);
    launch_dependent(cc_apply_scatter_kernel, gs, CC_APPLY_THREADS, 0, st, ctx->d_dev, ctx->tabs, lg);
    launch_dependent(cc_apply_cleanup_kernel, (unsigned)ctx->sm_count, CC_APPLY_THREADS, 0, st, ctx->d_dev, ctx->tabs, out);
    ctx->launches += 4;
    CC_CUDA(ctx, cudaGetLastError());
    return CC_OK;
}

// ---------------------------------------------------------- ring + persistent worker --

static inline u64 now_ns() {
    return (u64)std::chrono::duration_cast<std::chrono::nanoseconds>(std::chrono::steady_clock::now().time_since_epoch()).count();
}
static inline volatile u64* ring_tail(cc_ctx* c) { return c->ring_words + 0; }
static inline volatile u64* ring_completed(cc_ctx* c) { return c->ring_words + 8; }
static inline volatile u64* ring_heartbeat(cc_ctx* c) { return c->ring_words + 16; }

// Worker CTAs: the configured number; CC_WORKER_BLOCKS_ALL = as many as are co-resident; 0 = the default footprint
// CC_WORKER_BLOCKS_DEFAULT (about a ninth of the SMs: a bandwidth-bound application kernel next to an idle worker of
// that size keeps ~96 % of its throughput and a 256 MiB checkpoint task takes ~0.26 ms -- profiles/r02_bench_overlap.txt;
// the paper runs ONE block = 0.53 % of its SMs, which on B200 moves ~70 GB/s).
static uint32_t worker_block_count(cc_ctx* ctx, int bps) {
    const uint32_t max = (uint32_t)(bps * ctx->sm_count);
    if (ctx->cfg.worker_blocks == CC_WORKER_BLOCKS_ALL) return max;
    if (ctx->cfg.worker_blocks == 0) return CC_WORKER_BLOCKS_DEFAULT < max ? CC_WORKER_BLOCKS_DEFAULT : max;
    return ctx->cfg.worker_blocks;
}

extern "C" int32_t cc_worker_start(cc_ctx* ctx) {
    if (!ctx) return CC_ERR_INVALID;
    if (ctx->worker_running) return CC_ERR_WORKER;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    int coop = 0;
    CC_CUDA(ctx, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device));
    if (!coop) return CC_ERR_WORKER;
    const int threads = (int)ctx->cfg.worker_threads;
    int bps = 0;
    CC_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, cc_worker_kernel, threads, sizeof(cc_crc_smem)));
    if (bps < 1) return CC_ERR_WORKER;
    const uint32_t blocks = worker_block_count(ctx, bps);
    if (blocks > (uint32_t)(bps * ctx->sm_count)) return CC_ERR_INVALID;   // must all be co-resident (grid barrier)
    // reset barrier / doorbell state and the host-side ring words
    struct { u32 bar_count, bar_gen; u64 doorbell; } z = {0, 0, 0};
    CC_CUDA(ctx, cudaMemcpyAsync(&ctx->d_dev->bar_count, &z.bar_count, 4, cudaMemcpyHostToDevice, 0));
    CC_CUDA(ctx, cudaMemcpyAsync(&ctx->d_dev->bar_gen, &z.bar_gen, 4, cudaMemcpyHostToDevice, 0));
    CC_CUDA(ctx, cudaMemcpyAsync(&ctx->d_dev->doorbell, &z.doorbell, 8, cudaMemcpyHostToDevice, 0));
    CC_CUDA(ctx, cudaStreamSynchronize(0));
    memset(ctx->ring_results, 0, (size_t)ctx->cfg.ring_capacity * sizeof(cc_result));
    *ring_tail(ctx) = 0;
    *ring_completed(ctx) = 0;
    *ring_heartbeat(ctx) = 0;
    ctx->submitted = 0;
    std::atomic_thread_fence(std::memory_order_seq_cst);
    cc_ring_dev ring;
    ring.slots = ctx->ring_slots;
    ring.results = ctx->ring_results;
    ring.tail = (u64*)ring_tail(ctx);
    ring.completed = (u64*)ring_completed(ctx);
    ring.heartbeat = (u64*)ring_heartbeat(ctx);
    ring.capacity = ctx->cfg.ring_capacity;
    ring.backoff_ns = ctx->cfg.backoff_ns;
    ring.max_lifetime_ns = ctx->cfg.max_lifetime_ns;
    cc_dev* d = ctx->d_dev;
    cc_apply_tabs tabs = ctx->tabs;
    if (!ctx->apply_attached) memset(&tabs, 0, sizeof(tabs));
    void* args[] = {&d, &ring, &tabs};
    CC_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)cc_worker_kernel, dim3(blocks), dim3(threads), args,
                                             sizeof(cc_crc_smem), ctx->worker_stream));
    CC_CUDA(ctx, cudaEventRecord(ctx->worker_done, ctx->worker_stream));
    ctx->launches += 1;
    ctx->worker_running = true;
    ctx->worker_blocks_used = blocks;
    return CC_OK;
}

// Has the worker kernel left by itself (max_lifetime_ns expiry, a fault)?  Then nothing will ever complete again:
// mark it stopped so that cc_submit / cc_wait report CC_ERR_WORKER (or CC_ERR_CUDA) instead of spinning.
static int32_t worker_gone(cc_ctx* ctx) {
    if (!ctx->worker_running) return CC_ERR_WORKER;
    const cudaError_t q = cudaEventQuery(ctx->worker_done);
    if (q == cudaErrorNotReady) return CC_OK;
    ctx->worker_running = false;
    if (q != cudaSuccess) { ctx->last_cuda = (int)q; return CC_ERR_CUDA; }
    return CC_ERR_WORKER;
}

extern "C" int32_t cc_submit(cc_ctx* ctx, const cc_task* task, uint64_t* seq_out) {
    if (!ctx || !task) return CC_ERR_INVALID;
    if (!ctx->worker_running) return CC_ERR_WORKER;
    if (ctx->in_submit.exchange(1u, std::memory_order_acquire)) return CC_ERR_INVALID;   // a second producer is inside
    const u64 seq = ctx->submitted;
    const u64 done = __atomic_load_n(ctx->ring_words + 8, __ATOMIC_ACQUIRE);
    if (seq - done >= ctx->cfg.ring_capacity) {
        const int32_t g = worker_gone(ctx);          // full because the worker died?
        ctx->in_submit.store(0u, std::memory_order_release);
        return g != CC_OK ? g : CC_ERR_RING_FULL;
    }
    cc_task* slot = &ctx->ring_slots[seq & (ctx->cfg.ring_capacity - 1)];
    cc_task t = *task;
    t.seq = seq;
    memcpy(slot, &t, sizeof(t));                                         // write(slot, desc)
    __atomic_store_n(ctx->ring_words + 0, seq + 1, __ATOMIC_RELEASE);    // commit(slot): store-release
    ctx->submitted = seq + 1;
    if (seq_out) *seq_out = seq;
    ctx->in_submit.store(0u, std::memory_order_release);
    return CC_OK;
}

#if CC_BENCH_HOOKS
__global__ void cc_empty_kernel() {}

// Measurement hook for the comparison of PAPER.md Table 7 (L368-370: cudaLaunchKernel 7.6 us with a sync per launch,
// 2.5 us batched): mean ns per launch of an empty kernel on `stream`, (a) synchronising after every launch and
// (b) launching n back to back and synchronising once.  Must not be called while the worker is resident on every SM.
extern "C" int32_t cc_measure_launch_cost(cc_ctx* ctx, uint32_t n, void* stream, double* ns_sync, double* ns_batched) {
    if (!ctx || n == 0 || !ns_sync || !ns_batched) return CC_ERR_INVALID;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    for (int i = 0; i < 16; i++) cc_empty_kernel<<<1, 32, 0, st>>>();
    CC_CUDA(ctx, cudaStreamSynchronize(st));
    u64 t0 = now_ns();
    for (uint32_t i = 0; i < n; i++) {
        cc_empty_kernel<<<1, 32, 0, st>>>();
        CC_CUDA(ctx, cudaStreamSynchronize(st));
    }
    *ns_sync = (double)(now_ns() - t0) / n;
    t0 = now_ns();
    for (uint32_t i = 0; i < n; i++) cc_empty_kernel<<<1, 32, 0, st>>>();
    CC_CUDA(ctx, cudaStreamSynchronize(st));
    *ns_batched = (double)(now_ns() - t0) / n;
    ctx->launches += 2ull * n + 16;
    return CC_OK;
}

// Measurement hook: the host cost of cc_submit itself, without a language binding in the way (PAPER.md:L162,
// Table 7 "ring submit < 0.1 us").  Submits n CC_TASK_NOP tasks; only the cc_submit calls are inside the timed
// sections (when the ring is full the wait for a free slot is not).  Returns the mean ns per cc_submit.
extern "C" int32_t cc_measure_submit_cost(cc_ctx* ctx, uint32_t n, double* ns_per_submit) {
    if (!ctx || !ns_per_submit || n == 0) return CC_ERR_INVALID;
    if (!ctx->worker_running) return CC_ERR_WORKER;
    cc_task t;
    memset(&t, 0, sizeof(t));
    t.kind = CC_TASK_NOP;
    u64 total = 0, seq = 0;
    uint32_t done = 0;
    while (done < n) {
        const u64 room = ctx->cfg.ring_capacity - (ctx->submitted - __atomic_load_n(ctx->ring_words + 8, __ATOMIC_ACQUIRE));
        uint32_t burst = (uint32_t)(room < (n - done) ? room : (n - done));
        if (burst == 0) {
            if (cudaEventQuery(ctx->worker_done) != cudaErrorNotReady) return CC_ERR_WORKER;
            continue;
        }
        const u64 t0 = now_ns();
        for (uint32_t i = 0; i < burst; i++)
            if (cc_submit(ctx, &t, &seq) != CC_OK) return CC_ERR_RING_FULL;
        total += now_ns() - t0;
        done += burst;
    }
    cc_result r;
    int32_t rc = cc_wait(ctx, seq, 10ull * 1000000000ull, &r);
    if (rc != CC_OK) return rc;
    *ns_per_submit = (double)total / (double)n;
    return CC_OK;
}

#endif  // CC_BENCH_HOOKS

extern "C" int32_t cc_poll(cc_ctx* ctx, uint64_t seq, cc_result* out) {
    if (!ctx) return CC_ERR_INVALID;
    if (seq >= ctx->submitted) return CC_ERR_INVALID;
    cc_result* r = &ctx->ring_results[seq & (ctx->cfg.ring_capacity - 1)];
    const u64 sd = __atomic_load_n(&r->seq_done, __ATOMIC_ACQUIRE);
    if (sd != seq + 1) return sd > seq + 1 ? CC_ERR_INVALID : CC_PENDING;   // slot already reused: too late
    if (out) memcpy(out, r, sizeof(*r));
    return CC_OK;
}

extern "C" int32_t cc_wait(cc_ctx* ctx, uint64_t seq, uint64_t timeout_ns, cc_result* out) {
    const u64 t0 = now_ns();
    u64 next_check = t0 + 2000000ull;       // look at the worker kernel itself every 2 ms
    for (;;) {
        int32_t rc = cc_poll(ctx, seq, out);
        if (rc != CC_PENDING) return rc;
        const u64 now = now_ns();
        if (now - t0 > timeout_ns) return CC_ERR_TIMEOUT;
        if (now >= next_check) {
            const int32_t g = worker_gone(ctx);
            if (g != CC_OK) return cc_poll(ctx, seq, out) == CC_OK ? CC_OK : g;     // it may have finished this task last
            next_check = now + 2000000ull;
        }
#if defined(__x86_64__)
        __builtin_ia32_pause();
#endif
    }
}

extern "C" int32_t cc_peek_queue(cc_ctx* ctx, uint64_t* head, uint64_t* tail) {
    if (!ctx) return CC_ERR_INVALID;
    if (head) *head = __atomic_load_n(ctx->ring_words + 8, __ATOMIC_ACQUIRE);
    if (tail) *tail = ctx->submitted;
    return CC_OK;
}

extern "C" int32_t cc_worker_alive(cc_ctx* ctx) {
    if (!ctx || !ctx->worker_running) return 0;
    cudaSetDevice(ctx->device);
    if (cudaEventQuery(ctx->worker_done) != cudaErrorNotReady) return 0;    // kernel has left (or failed)
    const u64 hb0 = __atomic_load_n(ctx->ring_words + 16, __ATOMIC_ACQUIRE);
    const u64 t0 = now_ns();
    const struct timespec nap = {0, 20000};                                   // 20 us: the heartbeat moves every few us
    while (now_ns() - t0 < 1000000000ull) {
        if (__atomic_load_n(ctx->ring_words + 16, __ATOMIC_ACQUIRE) != hb0) return 1;
        nanosleep(&nap, nullptr);                                             // a dead worker costs a sleeping second, not a spinning core
    }
    return 0;
}

// Footprint of the persistent worker (Table 9: "1 block out of 188 SMs = 0.53 % of GPU resources"):
// CTAs (of the running worker, else what cc_worker_start would launch), threads per CTA, shared memory per CTA
// (static + dynamic), registers per thread, SMs of the device.
extern "C" int32_t cc_worker_footprint(cc_ctx* ctx, uint32_t* blocks, uint32_t* threads, uint32_t* smem_bytes, uint32_t* regs,
                                       uint32_t* sm_count) {
    if (!ctx) return CC_ERR_INVALID;
    CC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaFuncAttributes fa;
    CC_CUDA(ctx, cudaFuncGetAttributes(&fa, cc_worker_kernel));
    const int th = (int)ctx->cfg.worker_threads;
    uint32_t b = ctx->worker_blocks_used;
    if (!ctx->worker_running) {
        int bps = 0;
        CC_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, cc_worker_kernel, th, sizeof(cc_crc_smem)));
        b = worker_block_count(ctx, bps);
    }
    if (blocks) *blocks = b;
    if (threads) *threads = (uint32_t)th;
    if (smem_bytes) *smem_bytes = (uint32_t)(fa.sharedSizeBytes + sizeof(cc_crc_smem));
    if (regs) *regs = (uint32_t)fa.numRegs;
    if (sm_count) *sm_count = (uint32_t)ctx->sm_count;
    return CC_OK;
}

extern "C" int32_t cc_worker_stop(cc_ctx* ctx) {
    if (!ctx) return CC_ERR_INVALID;
    if (!ctx->worker_running) return CC_ERR_WORKER;
    ctx->in_submit.store(0u, std::memory_order_release);
    cudaSetDevice(ctx->device);
    cc_task t;
    memset(&t, 0, sizeof(t));
    t.kind = CC_TASK_EXIT;
    const u64 t0 = now_ns();
    bool sent = false;
    for (;;) {
        cudaError_t q = cudaEventQuery(ctx->worker_done);
        if (q == cudaSuccess) break;
        if (q != cudaErrorNotReady) { ctx->last_cuda = (int)q; ctx->worker_running = false; return CC_ERR_CUDA; }
        if (!sent && cc_submit(ctx, &t, nullptr) == CC_OK) sent = true;
        if (now_ns() - t0 > 10ull * 1000000000ull) return CC_ERR_TIMEOUT;
    }
    ctx->worker_running = false;
    return CC_OK;
}
