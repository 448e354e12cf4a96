// cc_tasks.cuh -- grid barrier and the classic (multi-phase) checkpoint of one region as ONE device function, shared by
// the persistent worker (cc_worker.cuh) and by the single-pass kernel's fallback (cc_pass_kernel in concordia.cu).
#pragma once
#include "cc_common.cuh"
#include "cc_ckpt.cuh"
#include "cc_mark.cuh"
#include "cc_rle.cuh"
#include "cc_pass.cuh"

// All blocks of the grid must be co-resident (cooperative launch).
__device__ __forceinline__ void cc_grid_barrier(cc_dev* dev, u32 nblocks, u32& gen) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&dev->bar_count, 1u) == nblocks - 1) {
            atomicExch(&dev->bar_count, 0u);
            __threadfence();
            atomicAdd(&dev->bar_gen, 1u);
        } else {
            while (ld_acquire_gpu_u32(&dev->bar_gen) == gen) __nanosleep(40);
        }
        __threadfence();
    }
    gen++;
    __syncthreads();
}


// a1 discovery -> a2 compaction -> [run ranking ->] a3-a5 record writer + commit, separated by grid barriers
// (PAPER.md:L259-264).  Discovery: compare (scan), the runtime's marks (optionally verified) or version counters
// (L257), or every page (base snapshot, L394).  Run-length records (L221) take three more phases.
__device__ __forceinline__ void cc_classic_checkpoint(cc_dev* dev, const cc_region_dev& r, cc_crc_smem* cs, const cc_pass_args& a,
                                                      cc_grid g, u32& gen, cc_result* out, bool init_tables) {
    const bool rle = a.run_pages > 1;
    const u32 final_mode = rle ? CC_MODE_SCAN_ONLY : CC_MODE_CHECKPOINT;
    switch (a.disc) {
    case CC_DISC_SCAN:
        cc_scan_phase<8>(r, g);
        cc_grid_barrier(dev, g.nblocks, gen);
        cc_compact_phase(r, &dev->log, final_mode, a.epoch, nullptr);
        break;
    case CC_DISC_MARKS:
    case CC_DISC_MARKS_VERIFY:
        cc_mark_load_phase(r, a.marks, g);
        cc_grid_barrier(dev, g.nblocks, gen);
        if (a.disc == CC_DISC_MARKS_VERIFY) {
            cc_compact_phase(r, &dev->log, CC_MODE_SCAN_ONLY, a.epoch, nullptr);
            cc_grid_barrier(dev, g.nblocks, gen);
            cc_mark_verify_phase(r, g);
            cc_grid_barrier(dev, g.nblocks, gen);
        }
        cc_compact_phase(r, &dev->log, final_mode, a.epoch, nullptr);
        break;
    case CC_DISC_VERSIONS:
        cc_mark_versions_phase(r, a.version, a.committed, g);
        cc_grid_barrier(dev, g.nblocks, gen);
        cc_compact_phase(r, &dev->log, final_mode, a.epoch, nullptr);
        break;
    default:
        cc_snapshot_plan_phase(r, &dev->log, a.epoch, g);
        break;
    }
    cc_grid_barrier(dev, g.nblocks, gen);
    if (rle) {
        cc_rle_starts_phase(r, a.run_pages, g);
        cc_grid_barrier(dev, g.nblocks, gen);
        cc_rle_rank_phase(r, &dev->log);
        cc_grid_barrier(dev, g.nblocks, gen);
        cc_rle_plan_phase(r, &dev->log, a.epoch, g);
        cc_grid_barrier(dev, g.nblocks, gen);
        cc_rle_gather_phase(r, dev, cs, g, out, a.kind, init_tables);
    } else {
        cc_gather_phase(r, dev, cs, g, out, a.kind, init_tables);
    }
    if ((a.disc == CC_DISC_MARKS || a.disc == CC_DISC_MARKS_VERIFY) && a.consume) {
        cc_grid_barrier(dev, g.nblocks, gen);
        cc_mark_finish_phase(r, a.marks, nullptr, nullptr, g);
    } else if (a.disc == CC_DISC_VERSIONS) {
        cc_grid_barrier(dev, g.nblocks, gen);
        cc_mark_finish_phase(r, nullptr, a.version, a.committed, g);
    }
}
