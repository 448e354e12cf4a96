// cc_batch.cuh -- one boundary, all regions ("At each NCCL or kernel
// boundary, a four-stage GPU-side pipeline executes" over the registered mutable regions, L217, L257).
// Every registered region that has a shadow is delta-checkpointed with the same epoch number, in
// ascending region_id order in the log, in FOUR launches whatever the number of regions:
//   scan-all    cc_scan_phase over every region (the grid strides over one region after the other)
//   rank-all    the ordered compaction of every region's bitmap (k per region); a small region is ranked
//               by ONE block (round-robin over the blocks), a large one by the whole grid
//   plan        one block, one thread per region slot: rank the regions by id, sizes in parallel, one thread
//               chains the log offset over the (<= 64) sizes in shared memory, plans written in parallel.
//               A region that does not fit is skipped whole (its own all-or-nothing rule), the ones after
//               it are still tried
//   gather-all  cc_gather_work over every region with no synchronisation in between; ONE completion for
//               the whole boundary: the last block appends every region's commit record, fences, publishes
//               the final offset once (a published offset means "everything before it is committed") and
//               fills the aggregated result.
// Same bytes as calling cc_checkpoint_delta region by region in ascending id order.
#pragma once
#include "cc_common.cuh"
#include "cc_ckpt.cuh"

#define CC_BATCH_SMALL_TILES 4u     // regions with at most this many compaction tiles are ranked by a single block

__device__ __forceinline__ bool cc_batch_takes_part(const cc_dev* dev, int s) {
    return dev->region_used[s] && dev->regions[s].shadow != nullptr;
}

// The regions' work items form ONE index space (region after region); warp w takes the global items
// w, w + nwarps, ...  A per-block table in shared memory (item count per region slot, built by one thread per
// slot) tells a warp which of its items fall into which region, so that it never touches a region it has no
// item in -- with many small regions the cost is the sum of the work, not a chain of per-region latencies.
struct cc_batch_tab {
    u64 n_items[CC_MAX_REGIONS];
    u64 cum[CC_MAX_REGIONS + 1];
    u32 mod[CC_MAX_REGIONS];            // cum[s] % nwarps: a warp's first item of a region is one subtraction away
};

// call with all threads of the block; n_items[] filled by threads < CC_MAX_REGIONS beforehand
__device__ __forceinline__ void cc_batch_tab_finish(cc_batch_tab* T, u64 nwarps) {
    __syncthreads();
    if (threadIdx.x == 0) {
        u64 c = 0;
        for (int s = 0; s < CC_MAX_REGIONS; s++) { T->cum[s] = c; c += T->n_items[s]; }
        T->cum[CC_MAX_REGIONS] = c;
    }
    __syncthreads();
    // one 64-bit remainder per slot and BLOCK, not per slot and warp (7,104 warps x 64 slots of software division were
    // most of the 38 M instructions cc_batch_scan_kernel executed on 48 small regions)
    if (threadIdx.x < CC_MAX_REGIONS) T->mod[threadIdx.x] = (u32)(T->cum[threadIdx.x] % nwarps);
    __syncthreads();
}

// first local item of region slot s for this warp (>= n_items[s] if none); warp < nwarps < 2^32
__device__ __forceinline__ u64 cc_batch_first(const cc_batch_tab* T, int s, u64 warp, u64 nwarps) {
    const u32 w = (u32)warp, m = T->mod[s];
    return w >= m ? (u64)(w - m) : (u64)(w + (u32)nwarps - m);
}

__device__ __forceinline__ void cc_batch_scan_phase(cc_dev* dev, cc_batch_tab* T, cc_grid g) {
    if (g.block == 0 && threadIdx.x == 0) {
        dev->batch.t_start_ns = globaltimer_ns();
        dev->batch.done = 0;
    }
    if (threadIdx.x < CC_MAX_REGIONS) {
        const int s = (int)threadIdx.x;
        u64 n = 0;
        if (cc_batch_takes_part(dev, s)) {
            const cc_region_dev& r = dev->regions[s];
            n = cc_scan_item_count<8>(r, g.nwarps());
            if (g.block == 0) {                             // open the region's compaction run (as cc_scan_phase does)
                r.hdr->t_start_ns = globaltimer_ns();
                r.hdr->ticket = 0;
                r.hdr->run_id = r.hdr->run_id + 1;
            }
        }
        T->n_items[s] = n;
    }
    cc_batch_tab_finish(T, g.nwarps());
    const u64 w = g.warp(), nw = g.nwarps();
    for (int s = 0; s < CC_MAX_REGIONS; s++) {
        if (T->n_items[s] == 0) continue;
        const u64 first = cc_batch_first(T, s, w, nw);
        if (first < T->n_items[s]) cc_scan_items<8>(dev->regions[s], first, nw);
    }
}

__device__ __forceinline__ void cc_batch_rank_phase(cc_dev* dev, u64 epoch, cc_grid g) {
    // which slots take part and how many compaction tiles they have: one thread per slot, in parallel (a block walking
    // the 64 slots one after the other paid 64 dependent round trips to global memory: 42 us for 48 small regions)
    __shared__ u32 s_tiles[CC_MAX_REGIONS];
    if (threadIdx.x < CC_MAX_REGIONS) {
        const int s = (int)threadIdx.x;
        u32 nt = 0;
        if (cc_batch_takes_part(dev, s))
            nt = (u32)((dev->regions[s].n_words + CC_COMPACT_TILE_WORDS - 1) / CC_COMPACT_TILE_WORDS);
        s_tiles[s] = nt;                                      // 0: takes no part
    }
    __syncthreads();
    u32 ordinal = 0;
    for (int s = 0; s < CC_MAX_REGIONS; s++) {
        const u32 nt = s_tiles[s];
        if (nt == 0) continue;
        const bool mine = nt > CC_BATCH_SMALL_TILES || (ordinal % g.nblocks) == g.block;
        ordinal++;
        if (mine) cc_compact_phase(dev->regions[s], &dev->log, CC_MODE_SCAN_ONLY, epoch, nullptr);
    }
}

// One block of at least CC_MAX_REGIONS threads.
__device__ __forceinline__ void cc_batch_plan_phase(cc_dev* dev, u64 epoch) {
    __shared__ u32 s_id[CC_MAX_REGIONS], s_order[CC_MAX_REGIONS], s_n;
    __shared__ u64 s_need[CC_MAX_REGIONS], s_W[CC_MAX_REGIONS];
    cc_batch_state* B = &dev->batch;
    const cc_log_dev* log = &dev->log;
    const u32 t = threadIdx.x;
    const bool part = t < CC_MAX_REGIONS && cc_batch_takes_part(dev, (int)t);
    if (t < CC_MAX_REGIONS) s_id[t] = part ? dev->regions[t].region_id : 0xFFFFFFFFu;
    if (t == 0) s_n = 0;
    __syncthreads();
    u32 k = 0;
    bool last_dirty = false;
    if (part) {
        const cc_region_dev& r = dev->regions[t];
        u32 rank = 0;
        for (u32 q = 0; q < CC_MAX_REGIONS; q++) rank += (s_id[q] < s_id[t]) ? 1u : 0u;     // ids are distinct
        s_order[rank] = t;
        atomicAdd(&s_n, 1u);
        k = r.hdr->k;
        last_dirty = k != 0 && r.D[k - 1] == (u32)(r.n_pages - 1);
        u64 need = 0;
        if (k) {
            need = (u64)k * (CC_RECORD_HEADER_BYTES + (u64)r.page_bytes) + CC_COMMIT_RECORD_BYTES;
            if (last_dirty) need -= (u64)r.page_bytes - page_len_dev(r, r.n_pages - 1);
        }
        s_need[t] = need;
    }
    __syncthreads();
    if (t == 0) {                       // the only sequential part: <= 64 additions in shared memory
        u64 W = log->W;
        const u64 W_begin = W;
        for (u32 i = 0; i < s_n; i++) {
            const u32 q = s_order[i];
            s_W[q] = W;
            if (s_need[q] != 0 && log->buf != nullptr && W + s_need[q] <= log->capacity) W += s_need[q];
        }
        B->W_final = W;
        B->bytes_total = W - W_begin;
        B->epoch = epoch;
        B->n_active = s_n;
        B->k_total = 0;
        B->status = CC_OK;
    }
    __syncthreads();
    if (part) {
        const cc_region_dev& r = dev->regions[t];
        cc_plan_checkpoint_at(r, log, s_W[t], CC_MODE_CHECKPOINT, epoch, k, last_dirty, false);
        atomicAdd(reinterpret_cast<unsigned long long*>(&B->k_total), (unsigned long long)k);
    }
    __shared__ int32_t s_status[CC_MAX_REGIONS];
    if (part) s_status[t] = dev->regions[t].hdr->status;    // (its own thread has just written it; read back in parallel)
    __syncthreads();
    if (t == 0) {                       // status of the lowest-id region that failed
        for (u32 i = 0; i < s_n; i++) {
            const int32_t st = s_status[s_order[i]];
            if (st != CC_OK) { B->status = st; break; }
        }
        __threadfence();
    }
}

// cs must already hold the CRC tables.
__device__ __forceinline__ void cc_batch_gather_phase(cc_dev* dev, cc_crc_smem* cs, cc_batch_tab* T, cc_grid g, cc_result* out,
                                                      u32 kind) {
    cc_batch_state* B = &dev->batch;
    if (threadIdx.x < CC_MAX_REGIONS) {
        const int s = (int)threadIdx.x;
        u64 n = 0;
        if (cc_batch_takes_part(dev, s)) n = (u64)dev->regions[s].hdr->k_eff * dev->regions[s].spp;
        T->n_items[s] = n;
    }
    cc_batch_tab_finish(T, g.nwarps());
    {
        const u64 w = g.warp(), nw = g.nwarps();
        for (int s = 0; s < CC_MAX_REGIONS; s++) {
            if (T->n_items[s] == 0) continue;
            const u64 first = cc_batch_first(T, s, w, nw);
            if (first < T->n_items[s]) cc_gather_items(dev->regions[s], dev, cs, first, nw);
        }
    }
    // ---- one completion for the whole boundary (same fence chain as cc_gather_complete: gpu-scope per block, ONE
    //      system-scope fence in the last block behind every commit record) ----
    __shared__ u32 s_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = (atomicAdd(&B->done, 1u) == g.nblocks - 1) ? 1u : 0u;
        if (s_last) __threadfence();
    }
    __syncthreads();
    if (!s_last) return;
    if (threadIdx.x < CC_MAX_REGIONS && cc_batch_takes_part(dev, (int)threadIdx.x))
        cc_gather_commit_record(dev->regions[threadIdx.x], dev);
    __syncthreads();
    if (threadIdx.x == 0) {
        cc_log_dev* log = &dev->log;
        B->done = 0;
        if (out) {
            out->n_dirty = B->k_total;
            out->bytes = B->bytes_total;
            out->log_offset_after = B->W_final;
            out->epoch = B->epoch;
            out->status = B->status;
            out->flags = kind;
            out->t_start_ns = B->t_start_ns;
            out->t_end_ns = globaltimer_ns();
        }
        __threadfence_system();
        if (B->bytes_total != 0) cc_log_publish_fenced(log, B->W_final);
        if (out) st_relaxed_sys_u64(&out->seq_done, 1ull);
    }
}
