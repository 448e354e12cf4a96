// cc_batch.cuh -- one boundary, all regions ("At each NCCL or kernel
// boundary, a four-stage GPU-side pipeline executes" over the registered mutable regions, L217, L257).
// Every registered region that has a shadow is delta-checkpointed with the same epoch number, in
// ascending region_id order in the log, in FOUR launches whatever the number of regions:
//   scan-all    cc_scan_phase over every region (the grid strides over one region after the other)
//   rank-all    the ordered compaction of every region's bitmap (k per region)
//   plan        one thread: ascending region_id, running log offset; a region that does not fit is
//               skipped whole (its own all-or-nothing rule), the ones after it are still tried
//   gather-all  cc_gather_phase over every region; a region's last block appends its commit record;
//               the last region to finish publishes the final offset ONCE (a published offset means
//               "everything before it is committed", so per-region publishes could not be reordered)
//               and fills the aggregated result.
// Same bytes as calling cc_checkpoint_delta region by region in ascending id order.
#pragma once
#include "cc_common.cuh"
#include "cc_ckpt.cuh"

__device__ __forceinline__ bool cc_batch_takes_part(const cc_dev* dev, int s) {
    return dev->region_used[s] && dev->regions[s].shadow != nullptr;
}

__device__ __forceinline__ void cc_batch_scan_phase(cc_dev* dev, cc_grid g) {
    if (g.block == 0 && threadIdx.x == 0) {
        dev->batch.t_start_ns = globaltimer_ns();
        dev->batch.done = 0;
    }
    for (int s = 0; s < CC_MAX_REGIONS; s++)
        if (cc_batch_takes_part(dev, s)) cc_scan_phase<8>(dev->regions[s], g);
}

__device__ __forceinline__ void cc_batch_rank_phase(cc_dev* dev, u64 epoch) {
    for (int s = 0; s < CC_MAX_REGIONS; s++)
        if (cc_batch_takes_part(dev, s)) cc_compact_phase(dev->regions[s], &dev->log, CC_MODE_SCAN_ONLY, epoch, nullptr);
}

// One thread.
__device__ __forceinline__ void cc_batch_plan_phase(cc_dev* dev, u64 epoch) {
    cc_batch_state* B = &dev->batch;
    const cc_log_dev* log = &dev->log;
    u64 W = log->W, k_total = 0;
    const u64 W_begin = W;
    int32_t first_bad = CC_OK;
    u32 n_active = 0, prev = 0;
    for (;;) {
        int best = -1;
        for (int s = 0; s < CC_MAX_REGIONS; s++)
            if (cc_batch_takes_part(dev, s) && dev->regions[s].region_id > prev &&
                (best < 0 || dev->regions[s].region_id < dev->regions[best].region_id))
                best = s;
        if (best < 0) break;
        const cc_region_dev& r = dev->regions[best];
        prev = r.region_id;
        n_active++;
        const u32 k = r.hdr->k;
        const bool last_dirty = k != 0 && r.D[k - 1] == (u32)(r.n_pages - 1);
        cc_plan_checkpoint_at(r, log, W, CC_MODE_CHECKPOINT, epoch, k, last_dirty, false);
        W += r.hdr->need;
        k_total += k;
        if (r.hdr->status != CC_OK && first_bad == CC_OK) first_bad = r.hdr->status;
    }
    B->W_final = W;
    B->k_total = k_total;
    B->bytes_total = W - W_begin;
    B->epoch = epoch;
    B->status = first_bad;
    B->n_active = n_active;
    __threadfence();
}

__device__ __forceinline__ void cc_batch_write_result(cc_dev* dev, cc_result* out, u32 kind) {
    const cc_batch_state* B = &dev->batch;
    if (!out) return;
    out->n_dirty = B->k_total;
    out->bytes = B->bytes_total;
    out->log_offset_after = B->W_final;
    out->epoch = B->epoch;
    out->status = B->status;
    out->flags = kind;
    out->t_start_ns = B->t_start_ns;
    out->t_end_ns = globaltimer_ns();
    __threadfence_system();
    st_release_sys_u64(&out->seq_done, 1ull);
}

// Called by the last block of a region's gather (one thread), after the region's commit record and a
// system-scope fence.  The last region to arrive publishes for the whole boundary.
__device__ __forceinline__ void cc_batch_region_done(cc_dev* dev, cc_result* out, u32 kind) {
    cc_batch_state* B = &dev->batch;
    __threadfence();
    if (atomicAdd(&B->done, 1u) != B->n_active - 1) return;
    __threadfence_system();
    cc_log_dev* log = &dev->log;
    if (B->bytes_total != 0) {
        if (log->committed_off) st_release_sys_u64(log->committed_off, B->W_final);
        log->W = B->W_final;
    }
    cc_batch_write_result(dev, out, kind);
}

__device__ __forceinline__ void cc_batch_gather_phase(cc_dev* dev, cc_crc_smem* cs, cc_grid g, cc_result* out, u32 kind) {
    if (dev->batch.n_active == 0) {
        if (g.block == 0 && threadIdx.x == 0) cc_batch_write_result(dev, out, kind);
        return;
    }
    for (int s = 0; s < CC_MAX_REGIONS; s++)
        if (cc_batch_takes_part(dev, s)) cc_gather_phase(dev->regions[s], dev, cs, g, out, kind, false, true);
}
