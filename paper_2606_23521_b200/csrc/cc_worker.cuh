// cc_worker.cuh -- a7: the persistent worker kernel and its host-mapped ring (PAPER.md:L119,
// L139-160 dispatch loop, L247-249 host-mapped memory + release/acquire protocol).
//
// Differences from the paper's worker, and why:
//   - many co-resident blocks (cooperative launch) instead of 1 block x 128 threads: one block
//     cannot move HBM bandwidth; FIFO, one task at a time across the whole grid because
//     checkpoint / restore order is semantic (reading #15);
//   - block 0 / thread 0 is the only thread that touches host memory: it polls the tail word,
//     copies the 64-byte descriptor to device memory and rings a device-memory doorbell that the
//     other blocks spin on (L2-resident); task phases are separated by a grid barrier;
//   - static switch instead of a JIT-filled function-pointer table.
#pragma once
#include "cc_common.cuh"
#include "cc_ckpt.cuh"
#include "cc_mark.cuh"
#include "cc_fused.cuh"
#include "cc_rle.cuh"
#include "cc_apply.cuh"
#include "cc_compactor.cuh"
#include "cc_batch.cuh"
#include "cc_pass.cuh"
#include "cc_small.cuh"
#include "cc_tasks.cuh"

struct cc_ring_dev {            // all pointers are pinned, device-mapped host memory
    cc_task* slots;             // capacity x 64 B
    cc_result* results;         // capacity x 64 B
    u64* tail;                  // host -> device: tasks submitted (store-release by the host)
    u64* completed;             // device -> host: tasks completed
    u64* heartbeat;             // device -> host: %globaltimer of the last poll
    u32 capacity;
    u32 backoff_ns;
    u64 max_lifetime_ns;
};

#if CC_BENCH_HOOKS
__device__ __forceinline__ void cc_task_mutate(const cc_region_dev& r, const cc_task& t, cc_grid g) {
    const u64 n_mut = t.arg0, A = t.arg1, h = t.arg2;
    for (u64 j = (u64)g.block * blockDim.x + threadIdx.x; j < n_mut; j += (u64)g.nblocks * blockDim.x) {
        const u64 page = (j * A + h) % r.n_pages;
        const u64 off = (h + j) % page_len_dev(r, page);
        r.base[page * r.page_bytes + off] ^= 0x5A;
    }
}
#else
#define CC_TASK_TEST_MUTATE 4u      // recognised only to be refused
#endif

#define CC_WORKER_MAX_THREADS 512
// Register budget of the resident kernel: 2 blocks of 512 threads per SM = 64 registers per thread, so that a worker
// block leaves half of an SM's register file (and 32 of its 64 warp slots) to the application's kernels -- or to a
// second worker block.  (-DCC_WORKER_MIN_BLOCKS=1 builds the 128-register variant for an A/B measurement.)
#ifndef CC_WORKER_MIN_BLOCKS
#define CC_WORKER_MIN_BLOCKS 2
#endif

// The applier's parse inside the worker: the one-block serial walk.  (The parallel parse of the host-launched path
// sizes its blocks for the candidate search and the epoch walks; the worker's blocks are wider and its logs -- one
// restore per recovery -- do not justify a second instantiation in the resident kernel.)
__device__ __forceinline__ void cc_worker_parse(cc_dev* dev, const cc_apply_tabs& tabs, const u8* log, u64 n, cc_grid g, u32& gen) {
    if (g.block == 0) cc_apply_parse_phase(dev, tabs, log, n, true);
    cc_grid_barrier(dev, g.nblocks, gen);
}

// The recovery-side tasks are cold: kept out of line so that their registers do not weigh on the
// checkpoint tasks of the dispatch loop.
__device__ __noinline__ void cc_worker_restore_task(cc_dev* dev, const cc_apply_tabs& tabs, cc_crc_smem* cs,
                                                    const cc_task& task, cc_grid g, u32& gen) {
    const u8* log = reinterpret_cast<const u8*>(task.arg0);
    cc_worker_parse(dev, tabs, log, task.arg1, g, gen);
    cc_apply_validate_phase(dev, tabs, cs, log, g, false);
    cc_grid_barrier(dev, g.nblocks, gen);
    cc_apply_latest_phase(dev, tabs, g);
    cc_grid_barrier(dev, g.nblocks, gen);
    cc_apply_scatter_phase(dev, tabs, log, g);
    cc_grid_barrier(dev, g.nblocks, gen);
    cc_apply_cleanup_phase(dev, tabs, g, nullptr, task.kind);
}

__device__ __noinline__ void cc_worker_compact_task(cc_dev* dev, const cc_apply_tabs& tabs, cc_crc_smem* cs,
                                                    const cc_task& task, cc_grid g, u32& gen) {
    const u8* in = reinterpret_cast<const u8*>(task.arg0);
    u8* outl = reinterpret_cast<u8*>(task.arg2);
    cc_worker_parse(dev, tabs, in, task.arg1, g, gen);
    cc_apply_validate_phase(dev, tabs, cs, in, g, false);
    cc_grid_barrier(dev, g.nblocks, gen);
    cc_compactor_mark_phase(dev, tabs, g);
    cc_grid_barrier(dev, g.nblocks, gen);
    cc_compactor_rank_phase(dev);
    cc_grid_barrier(dev, g.nblocks, gen);
    if (g.block == 0) cc_compactor_plan_phase(dev, task.arg3);
    cc_grid_barrier(dev, g.nblocks, gen);
    cc_compactor_copy_phase(dev, tabs, cs, in, outl, g);
    cc_grid_barrier(dev, g.nblocks, gen);
    cc_compactor_cleanup_phase(dev, tabs, g, nullptr, task.kind);
}

// One checkpoint of one region: the single pass (CC_TASKF_FUSED, when the worst case fits behind the write offset) or
// the classic phases -- the same device code as the host-launched calls.  Out of line, like the recovery-side
// tasks below: the dispatch loop stays small and every task body gets the register file to itself.
__device__ __noinline__ void cc_worker_ckpt_task(cc_dev* dev, const cc_region_dev& r, cc_crc_smem* cs, u32* s_crc_ready,
                                                 cc_small_smem* s_small, const cc_task& task, u64 t_start,
                                                 cc_grid g, u32& gen) {
    cc_pass_args a;
    a.epoch = task.epoch; a.kind = task.kind; a.run_pages = 0; a.marks = nullptr; a.consume = 0;
    a.version = nullptr; a.committed = nullptr; a.disc = CC_DISC_SCAN;
    if (task.kind == CC_TASK_DELTA_CKPT) {
        if (task.flags & CC_TASKF_RLE) a.run_pages = (u32)task.arg0;
    } else if (task.kind == CC_TASK_MARKED_CKPT) {
        a.disc = (task.arg1 & CC_MARK_VERIFY) ? CC_DISC_MARKS_VERIFY : CC_DISC_MARKS;
        a.marks = reinterpret_cast<u32*>(task.arg0);
        a.consume = (task.arg1 & CC_MARK_CONSUME) ? 1u : 0u;
    } else if (task.kind == CC_TASK_VERSION_CKPT) {
        a.disc = CC_DISC_VERSIONS;
        a.version = reinterpret_cast<const u64*>(task.arg0);
        a.committed = reinterpret_cast<u64*>(task.arg1);
    } else a.disc = CC_DISC_ALL;
    const u64 W0 = dev->log.W;
    const bool single = (task.flags & CC_TASKF_FUSED) && cc_pass_supported(r.n_pages, a.run_pages) &&
                        dev->log.buf != nullptr && W0 + cc_pass_worst_bytes(r) <= dev->log.capacity;
    if (single) {
        if (g.block == 0 && threadIdx.x == 0) r.hdr->t_start_ns = t_start;
        const u32 TP = cc_pass_tile_pages(r, a.run_pages, g.nwarps());
        cc_pass_tiles(r, dev, cs, s_crc_ready, a, TP, W0, g);
        if (g.block == 0 && threadIdx.x == 0) CC_TRACE(dev, 11);
        cc_grid_barrier(dev, g.nblocks, gen);                 // (gpu-scope fences: every block's record bytes are behind block 0 now)
        if (g.block == 0 && threadIdx.x == 0) CC_TRACE(dev, 12);
        if (g.block == 0 && threadIdx.x < 32) cc_pass_commit(r, dev, nullptr, task.kind, threadIdx.x);   // ... and its ONE system-scope fence
        if (g.block == 0 && threadIdx.x == 0) CC_TRACE(dev, 13);
    } else if (a.disc == CC_DISC_SCAN && a.run_pages <= 1 && cc_small_supported(r.n_words)) {
        // small region, one record per page: scan, one rendezvous, every block ranks the bitmap by itself (cc_small.cuh)
        cc_small_checkpoint(dev, r, cs, s_small, task.epoch, task.kind, g, gen, nullptr, false);
        if (g.block == 0 && threadIdx.x == 0) r.hdr->t_start_ns = t_start;
    } else {
        cc_classic_checkpoint(dev, r, cs, a, g, gen, nullptr, false);
    }
}

__device__ __noinline__ void cc_worker_ckpt_all_task(cc_dev* dev, cc_crc_smem* cs, cc_batch_tab* btab, const cc_task& task,
                                                     cc_grid g, u32& gen) {
    cc_batch_scan_phase(dev, btab, g);
    cc_grid_barrier(dev, g.nblocks, gen);
    cc_batch_rank_phase(dev, task.epoch, g);
    cc_grid_barrier(dev, g.nblocks, gen);
    if (g.block == 0) cc_batch_plan_phase(dev, task.epoch);
    cc_grid_barrier(dev, g.nblocks, gen);
    cc_batch_gather_phase(dev, cs, btab, g, nullptr, task.kind);
}

__global__ void __launch_bounds__(CC_WORKER_MAX_THREADS, CC_WORKER_MIN_BLOCKS)
cc_worker_kernel(cc_dev* dev, cc_ring_dev ring, cc_apply_tabs tabs) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cc_crc_smem* cs = reinterpret_cast<cc_crc_smem*>(smem_raw);
    __shared__ __align__(16) cc_task s_task;
    __shared__ cc_batch_tab s_btab;
    __shared__ cc_small_smem s_small;
    __shared__ u32 s_crc_ready;             // the CRC tables are filled once, at kernel start: always "ready"
    if (threadIdx.x == 0) s_crc_ready = 2u;
    const cc_grid g = cc_hw_grid();
    u32 gen = ld_acquire_gpu_u32(&dev->bar_gen);
    u64 head = 0;       // ring sequence number of the next task (meaningful in the leader thread only)
    u64 gseq = 0;       // number of grid-wide tasks so far = doorbell value already consumed
    const u64 t0 = globaltimer_ns();
    cc_crc_smem_init(cs, &dev->crc);

    for (;;) {
        // ---- leader: poll the host-mapped tail, fetch descriptors.  NOP and LOG_RESET need no grid:
        //      the leader completes them on the spot; anything else is handed to all blocks through
        //      the device-memory doorbell ----
        if (g.block == 0 && threadIdx.x == 0) {
            for (;;) {
                bool expired = false;
                u32 spins = 0;
                while (ld_acquire_sys_u64(ring.tail) <= head) {
                    const u64 now = globaltimer_ns();
                    if ((spins++ & 15u) == 0) *reinterpret_cast<volatile u64*>(ring.heartbeat) = now;
                    if (now - t0 > ring.max_lifetime_ns) { expired = true; break; }
                    __nanosleep(ring.backoff_ns);
                }
                cc_task t;
                if (expired) {
                    t.kind = CC_TASK_EXIT; t.region_id = 0; t.flags = 1; t.version = 0; t.seq = ~0ull;
                    t.epoch = 0; t.arg0 = t.arg1 = t.arg2 = t.arg3 = 0;
                } else {
                    // four independent 16-byte system-scope loads (one host-link round trip); they are
                    // ordered after the acquire of the tail word
                    const char* src = reinterpret_cast<const char*>(&ring.slots[head & (ring.capacity - 1)]);
                    uint4 q[4];
#pragma unroll
                    for (int i = 0; i < 4; i++) q[i] = ld_relaxed_sys_v4(src + 16 * i);
                    t = *reinterpret_cast<cc_task*>(q);
                }
                if (t.kind == CC_TASK_NOP || t.kind == CC_TASK_LOG_RESET) {
                    const u64 ts = globaltimer_ns();
                    if (t.kind == CC_TASK_LOG_RESET) cc_log_rewind(&dev->log);
                    cc_result* out = &ring.results[t.seq & (ring.capacity - 1)];
                    out->n_dirty = 0; out->bytes = 0; out->log_offset_after = dev->log.W; out->epoch = t.epoch;
                    out->status = CC_OK; out->flags = t.kind; out->t_start_ns = ts; out->t_end_ns = globaltimer_ns();
                    st_relaxed_sys_u64(ring.completed, t.seq + 1);     // a counter only; results are read through seq_done
                    st_release_sys_u64(&out->seq_done, t.seq + 1);     // release: every field above is visible first
                    head++;
                    continue;
                }
                dev->cur_task = t;
                __threadfence();
                st_release_gpu_u64(&dev->doorbell, gseq + 1);
                break;
            }
        }
        // ---- everyone: wait for the doorbell ----
        if (threadIdx.x == 0) {
            while (ld_acquire_gpu_u64(&dev->doorbell) <= gseq) __nanosleep(ring.backoff_ns < 200 ? ring.backoff_ns : 200);
            __threadfence();
            const uint4* ct = reinterpret_cast<const uint4*>(&dev->cur_task);
            uint4* st = reinterpret_cast<uint4*>(&s_task);
#pragma unroll
            for (int i = 0; i < 4; i++) st[i] = __ldcg(ct + i);
        }
        __syncthreads();
        const cc_task task = s_task;
        const u64 t_start = globaltimer_ns();
        if (task.kind == CC_TASK_EXIT) break;

        int32_t status = CC_OK;
        int slot = -1;
        const bool is_ckpt = task.kind == CC_TASK_DELTA_CKPT || task.kind == CC_TASK_MARKED_CKPT ||
                             task.kind == CC_TASK_VERSION_CKPT || task.kind == CC_TASK_SNAPSHOT;
        if (is_ckpt || task.kind == CC_TASK_TEST_MUTATE) {
            slot = cc_find_slot(dev, task.region_id);
            if (slot < 0) status = CC_ERR_NOT_REGISTERED;
            else if (dev->regions[slot].shadow == nullptr &&
                     (task.kind == CC_TASK_DELTA_CKPT || (task.kind == CC_TASK_MARKED_CKPT && (task.arg1 & CC_MARK_VERIFY))))
                status = CC_ERR_INVALID;
            if (task.kind == CC_TASK_MARKED_CKPT && (task.arg0 == 0 || (task.arg0 & 3))) status = CC_ERR_INVALID;
            if (slot >= 0 && task.kind == CC_TASK_DELTA_CKPT && (task.flags & CC_TASKF_RLE) &&
                (task.arg0 == 0 || task.arg0 > 0xFFFFFFFFull / dev->regions[slot].page_bytes))
                status = CC_ERR_INVALID;
            if (task.kind == CC_TASK_VERSION_CKPT && (task.arg0 == 0 || task.arg1 == 0 || ((task.arg0 | task.arg1) & 7)))
                status = CC_ERR_INVALID;
        }
        // recovery-side tasks: the applier tables must be attached (cc_apply_attach before cc_worker_start) and the
        // log pointers non-null and 16-byte aligned -- same checks as the host-launched cc_apply_log / cc_compact_log
        if (task.kind == CC_TASK_RESTORE || task.kind == CC_TASK_COMPACT_LOG) {
            if (tabs.max_records == 0 || task.arg0 == 0 || (task.arg0 & 15)) status = CC_ERR_INVALID;
            if (task.kind == CC_TASK_COMPACT_LOG) {
                if (task.arg2 == 0 || (task.arg2 & 15)) status = CC_ERR_INVALID;
                else if (task.arg0 < task.arg2 + task.arg3 && task.arg2 < task.arg0 + task.arg1) status = CC_ERR_INVALID;   // overlap
            }
        }
        if (status == CC_OK) {
            switch (task.kind) {
            case CC_TASK_DELTA_CKPT:
            case CC_TASK_MARKED_CKPT:
            case CC_TASK_VERSION_CKPT:
            case CC_TASK_SNAPSHOT:
                cc_worker_ckpt_task(dev, dev->regions[slot], cs, &s_crc_ready, &s_small, task, t_start, g, gen);
                break;
            case CC_TASK_CKPT_ALL:
                cc_worker_ckpt_all_task(dev, cs, &s_btab, task, g, gen);
                break;
            case CC_TASK_COMPACT_LOG:
                cc_worker_compact_task(dev, tabs, cs, task, g, gen);
                break;
            case CC_TASK_RESTORE:
                cc_worker_restore_task(dev, tabs, cs, task, g, gen);
                break;
            case CC_TASK_TEST_MUTATE:
#if CC_BENCH_HOOKS
                cc_task_mutate(dev->regions[slot], task, g);
#else
                status = CC_ERR_INVALID;
#endif
                break;
            default:
                break;
            }
        }
        // ---- end of task: everyone done, leader publishes the completion ----
        cc_grid_barrier(dev, g.nblocks, gen);
        if (g.block == 0 && threadIdx.x == 0) {
            cc_result* out = &ring.results[task.seq & (ring.capacity - 1)];
            u64 n_dirty = 0, bytes = 0, off_after = dev->log.W, ep = task.epoch;
            if (status == CC_OK && is_ckpt) {
                const cc_ws_hdr* h = dev->regions[slot].hdr;
                n_dirty = h->k; bytes = h->need; status = h->status;
            } else if (status == CC_OK && task.kind == CC_TASK_CKPT_ALL) {
                const cc_batch_state* B = &dev->batch;
                n_dirty = B->k_total; bytes = B->bytes_total; off_after = B->W_final; status = B->status;
            } else if (status == CC_OK && task.kind == CC_TASK_COMPACT_LOG) {
                const cc_compactor_state* C = &dev->compactor;
                n_dirty = C->n_out; bytes = C->bytes_out; off_after = dev->apply.consumed;
                ep = C->n_regions_out; status = C->status;
            } else if (status == CC_OK && task.kind == CC_TASK_RESTORE) {
                const cc_apply_state* A = &dev->apply;
                n_dirty = A->n_commit_recs; bytes = A->consumed; off_after = A->consumed;
                ep = A->n_commit_epochs; status = A->status;
            }
            out->n_dirty = n_dirty; out->bytes = bytes; out->log_offset_after = off_after; out->epoch = ep;
            out->status = status; out->flags = task.kind;
            out->t_start_ns = t_start; out->t_end_ns = globaltimer_ns();
            st_relaxed_sys_u64(ring.completed, task.seq + 1);
            st_release_sys_u64(&out->seq_done, task.seq + 1);
        }
        head++;
        gseq++;
    }
    // exit: the leader acknowledges the EXIT task (if it came from the host) and stamps the heartbeat
    if (g.block == 0 && threadIdx.x == 0) {
        const cc_task t = s_task;
        if (t.seq != ~0ull) {
            cc_result* out = &ring.results[t.seq & (ring.capacity - 1)];
            out->n_dirty = 0; out->bytes = 0; out->log_offset_after = dev->log.W; out->epoch = 0;
            out->status = CC_OK; out->flags = CC_TASK_EXIT; out->t_start_ns = globaltimer_ns(); out->t_end_ns = out->t_start_ns;
            st_relaxed_sys_u64(ring.completed, t.seq + 1);
            st_release_sys_u64(&out->seq_done, t.seq + 1);
        }
    }
}
