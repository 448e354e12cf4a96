// cc_small.cuh -- the low-latency checkpoint of a region whose dirty bitmap one block can rank by itself
// (<= CC_SMALL_MAX_WORDS bitmap words = 131,072 pages): a1 scan, a2 ranking, a3-a5 record writer and a4 commit in ONE
// launch with ONE grid-wide rendezvous (L100 / Table 6 "cost flat in the dirty count").
//
// Where the time of a small checkpoint goes (64 MiB, 1 % dirty: 55 us of device time as three kernels, 21 us of which is
// the HBM time of the scan itself) is launch gaps, the compaction kernel's ticket / look-back machinery for a 2 KiB
// bitmap, a chain of dependent cold loads per record and system-scope fences.  Here
//   scan      every warp compares 4 KiB segments (page-granular items with early-out when there are pages enough) and sets
//             bits of the workspace bitmap -- the same loop as cc_scan_kernel;
//   meet      one grid barrier (all blocks co-resident: cooperative launch / the resident worker); a block fills its
//             CRC tables between arriving and waiting;
//   rank      EVERY block reads the whole bitmap (a few KiB out of L2) and ranks it by itself: per-thread popcounts, one
//             block-wide exclusive scan, the per-thread offsets kept in shared memory.  Record i's page is then found
//             by a search in shared memory plus one 64-byte look at the bitmap: no dirty list has to be produced
//             first and waited for (one block still writes D[] for cc_dirty_list);
//   write     (record, 4 KiB segment) items round-robin over all warps -- cc_gather_segment, the same record writer;
//   commit    every block counts itself out (gpu-scope); the last one clears the bitmap, appends the commit record, fills
//             the result, executes the call's one system-scope fence and publishes (L263).
// Record kind: one record per page; discovery: compare.  Everything else takes cc_pass.cuh / the phases.
#pragma once
#include "cc_common.cuh"
#include "cc_crc.cuh"
#include "cc_ckpt.cuh"

#define CC_SMALL_MAX_WORDS 4096u            // bitmap words (32 pages each) a block ranks by itself
#define CC_SMALL_MAX_THREADS 512u

struct cc_small_smem {
    u32 excl[CC_SMALL_MAX_THREADS];         // records before thread t's words
    u32 warp_tot[CC_SMALL_MAX_THREADS / 32];
    u32 last_dirty, is_last;
};

__host__ __device__ __forceinline__ bool cc_small_supported(u64 n_words) { return n_words <= CC_SMALL_MAX_WORDS; }

// bitmap words per thread: a multiple of 4 (16-byte loads), so that blockDim threads cover all n_words
__device__ __forceinline__ u32 cc_small_wpt(const cc_region_dev& r) {
    const u32 per4 = (u32)((r.n_words + 4ull * blockDim.x - 1) / (4ull * blockDim.x));
    return 4u * (per4 ? per4 : 1u);
}

__device__ __forceinline__ uint4 ld_relaxed_gpu_v4(const void* p) {
    uint4 r;
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ u32 ld_relaxed_gpu_u32(const u32* p) {
    u32 v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// The page of record i (warp-uniform i; every lane gets the answer).  excl[] ascending; thread t owns bitmap words
// [t * wpt, (t + 1) * wpt).
__device__ __forceinline__ u32 cc_small_select(const cc_region_dev& r, const cc_small_smem* S, u32 wpt, u32 padded_words, u32 i, u32 lane) {
    u32 lo = 0, hi = blockDim.x;            // largest t with excl[t] <= i
    while (hi - lo > 1) {
        const u32 mid = (lo + hi) >> 1;
        if (S->excl[mid] <= i) lo = mid; else hi = mid;
    }
    const u32 t = lo;
    u32 rem = i - S->excl[t];
    u32 page = 0;
    for (u32 w0 = 0; w0 < wpt; w0 += 32) {                 // (wpt <= 16 with 256 threads: one round)
        const u32 wi = t * wpt + w0 + lane;
        const u32 w = (w0 + lane < wpt && wi < padded_words) ? ld_relaxed_gpu_u32(&r.bitmap[wi]) : 0u;
        const u32 c = __popc(w);
        u32 inc = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u32 n = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= (u32)o) inc += n;
        }
        const u32 total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        if (rem < total) {
            const u32 hit = __ballot_sync(0xFFFFFFFFu, rem < inc);       // first lane whose inclusive count exceeds rem
            const u32 src = (u32)__ffs(hit) - 1u;
            const u32 bit = __fns(w, 0, (int)(rem - (inc - c)) + 1);     // (meaningful in lane src)
            page = __shfl_sync(0xFFFFFFFFu, (wi << 5) + bit, src);
            break;
        }
        rem -= total;
    }
    return page;
}

// Everything behind the scan: rank, write, commit.  All blocks of the grid call it once the bitmap is complete (behind the
// rendezvous of cc_small_checkpoint, or as a kernel of its own behind cc_scan_kernel: cc_small_tail_kernel).
// tables_ready: cs already holds the CRC tables; otherwise a block fills them once it knows that it has records to write.
__device__ __forceinline__ void cc_small_tail(cc_dev* dev, const cc_region_dev& r, cc_crc_smem* cs, cc_small_smem* S, u64 epoch,
                                              u32 kind, cc_grid g, cc_result* out, bool tables_ready) {
    const u32 tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5;
    cc_ws_hdr* h = r.hdr;
    cc_log_dev* log = &dev->log;
    const u64 W0 = log->W;
    const u64 log_cap = log->capacity;
    const bool have_log = log->buf != nullptr;
    const u64 last_page = r.n_pages - 1;
    if (tid == 0) S->last_dirty = 0;
    __syncthreads();
    // ---- rank: every block, the whole bitmap ----
    const u32 wpt = cc_small_wpt(r);
    const u32 padded_words = (u32)((r.n_words + CC_COMPACT_TILE_WORDS - 1) / CC_COMPACT_TILE_WORDS * CC_COMPACT_TILE_WORDS);
    u32 cnt = 0;
    for (u32 q = 0; q < wpt; q += 4) {
        const u32 wi = tid * wpt + q;
        if (wi < padded_words) {
            const uint4 w = ld_relaxed_gpu_v4(&r.bitmap[wi]);
            cnt += __popc(w.x) + __popc(w.y) + __popc(w.z) + __popc(w.w);
            if ((u32)(last_page >> 7) == (wi >> 2)) {            // this 16-byte group holds the region's last page
                const u32 sel = (u32)(last_page >> 5) & 3u;
                const u32 lw = sel == 0 ? w.x : sel == 1 ? w.y : sel == 2 ? w.z : w.w;
                if ((lw >> (last_page & 31u)) & 1u) S->last_dirty = 1;
            }
        }
    }
    u32 inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u32 n = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= (u32)o) inc += n;
    }
    if (lane == 31) S->warp_tot[wid] = inc;
    const u32 my_excl_in_warp = inc - cnt;
    __syncthreads();
    u32 warp_base = 0, k = 0;
    for (u32 w = 0; w < (blockDim.x >> 5); w++) {
        const u32 v = S->warp_tot[w];
        if (w < wid) warp_base += v;
        k += v;
    }
    const u32 my_excl = warp_base + my_excl_in_warp;
    S->excl[tid] = my_excl;
    // the plan, identical in every block: record count, byte need, all-or-nothing log-full decision (reading #10)
    const bool last_dirty = S->last_dirty != 0;
    u64 need = (u64)k * (CC_RECORD_HEADER_BYTES + (u64)r.page_bytes) + CC_COMMIT_RECORD_BYTES;
    if (last_dirty) need -= (u64)r.page_bytes - page_len_dev(r, last_page);
    const bool fits = k != 0 && have_log && W0 + need <= log_cap;
    const u32 k_eff = fits ? k : 0u;
    __syncthreads();
    // ---- write: (record, segment) items round-robin over the grid's warps ----
    {
        const u32 spp = r.spp;
        const u64 n_items = (u64)k_eff * spp;
        if (!tables_ready && (u64)g.block * (blockDim.x >> 5) < n_items) cc_crc_smem_init(cs, &dev->crc);   // (block-uniform)
        for (u64 item = g.warp(); item < n_items; item += g.nwarps()) {
            u32 i, c;
            if (r.spp_shift >= 0) { i = (u32)(item >> r.spp_shift); c = (u32)(item & (spp - 1)); }
            else { i = (u32)(item / spp); c = (u32)(item - (u64)i * spp); }
            const u32 p = cc_small_select(r, S, wpt, padded_words, i, lane);
            cc_gather_segment(r, dev, cs, W0, i, c, p, lane);
        }
    }
    // ---- D[] for cc_dirty_list (the grid's last block: round-robin items reach it last; nobody inside this call reads D) ----
    if (g.block == g.nblocks - 1 && cnt != 0) {
        u32 pos = my_excl;
        for (u32 q = 0; q < wpt; q++) {
            const u32 wi = tid * wpt + q;
            u32 w = wi < padded_words ? ld_relaxed_gpu_u32(&r.bitmap[wi]) : 0u;
            while (w) {
                const u32 bit = (u32)__ffs(w) - 1u;
                w &= w - 1;
                r.D[pos++] = (wi << 5) + bit;
            }
        }
    }
    // ---- commit: every block counts out (all of them read the bitmap); the last one finishes the call ----
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        const u32 last = (atomicAdd(&h->gather_done, 1u) == g.nblocks - 1) ? 1u : 0u;
        if (last) __threadfence();
        S->is_last = last;
    }
    __syncthreads();
    if (!S->is_last) return;
    if (cnt != 0) {
        for (u32 q = 0; q < wpt; q += 4) {
            const u32 wi = tid * wpt + q;
            if (wi < padded_words) *reinterpret_cast<uint4*>(&r.bitmap[wi]) = make_uint4(0, 0, 0, 0);
        }
    }
    if (tid == 0) {
        CC_TRACE(dev, 12);
        cc_plan_checkpoint_at(r, log, W0, CC_MODE_CHECKPOINT, epoch, k, last_dirty, false);
        const u64 W_after = cc_gather_commit_record(r, dev);
        if (out) {
            out->n_dirty = k;
            out->bytes = h->need;
            out->log_offset_after = W_after;
            out->epoch = epoch;
            out->status = h->status;
            out->flags = kind;
            out->t_start_ns = h->t_start_ns;
            out->t_end_ns = globaltimer_ns();
        }
        __threadfence_system();             // the call's ONE system-scope fence
        if (k_eff != 0) cc_log_publish_fenced(log, W_after);
        if (out) st_relaxed_sys_u64(&out->seq_done, 1ull);
        CC_TRACE(dev, 13);
    }
}

// One launch: scan, ONE grid-wide rendezvous (all blocks co-resident: cooperative launch / the resident worker; a block
// fills its CRC tables while it waits), then cc_small_tail.  gen: the caller's grid-barrier generation (cc_tasks.cuh),
// advanced by one.
__device__ __forceinline__ void cc_small_checkpoint(cc_dev* dev, const cc_region_dev& r, cc_crc_smem* cs, cc_small_smem* S, u64 epoch,
                                                    u32 kind, cc_grid g, u32& gen, cc_result* out, bool init_tables) {
    const u32 tid = threadIdx.x;
    if (g.block == 0 && tid == 0) { r.hdr->t_start_ns = globaltimer_ns(); CC_TRACE(dev, 10); }
    cc_scan_items<8>(r, g.warp(), g.nwarps());
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(&dev->bar_count, 1u) == g.nblocks - 1) {
            atomicExch(&dev->bar_count, 0u);
            __threadfence();
            atomicAdd(&dev->bar_gen, 1u);
        }
    }
    if (init_tables) cc_crc_smem_init(cs, &dev->crc);
    if (tid == 0) {
        while (ld_acquire_gpu_u32(&dev->bar_gen) == gen) __nanosleep(32);
        __threadfence();
    }
    gen++;
    __syncthreads();
    if (g.block == 0 && tid == 0) CC_TRACE(dev, 11);
    cc_small_tail(dev, r, cs, S, epoch, kind, g, out, true);
}
