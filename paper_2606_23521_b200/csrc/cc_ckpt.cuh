// cc_ckpt.cuh -- the checkpoint direction: a1 scan, a2 compaction, a3-a5 gather + CRC + commit +
// shadow update.  Device functions over a virtual grid so that the
// host-launched kernels and the persistent worker run the very same code.
#pragma once
#include "cc_common.cuh"
#include "cc_crc.cuh"

// ------------------------------------------------------------------------- a1: scan --
// dirty[p] = any byte of cur page p differs from shadow page p.
// One warp compares 4 KiB segments: each lane issues 8 + 8 independent 16-byte streaming loads (cur, shadow),
// XOR/ORs them, the warp votes.  A work item is a whole page when there are pages enough to keep every warp busy
// (else a single segment): the warp walks the page's segments in order and STOPS at the first one that differs
// (per-page early-out: the rest of a dirty page is not read -- the gather reads it anyway), then lane 0 sets the
// page's bit in the bitmap.  The bitmap is all-zero on entry (the compaction clears what it consumes).
// Items first, first + step, ... of the region (the caller decides which warp takes which items).
// segments per work item for a grid of `nwarps` warps: the whole page if that still leaves >= 4 items per warp, else
// halved until it does (1 when the page's segment count is not a power of two)
template <int U>
__device__ __forceinline__ u32 cc_scan_group(const cc_region_dev& r, u64 nwarps) {
    const u32 spp = (r.page_bytes + 512u * U - 1) / (512u * U);
    if (spp & (spp - 1)) return 1;
    u32 G = spp;
    while (G > 1 && r.n_pages * (u64)(spp / G) < 4 * nwarps) G >>= 1;
    return G;
}
template <int U>
__device__ __forceinline__ u64 cc_scan_item_count(const cc_region_dev& r, u64 nwarps) {
    const u32 spp = (r.page_bytes + 512u * U - 1) / (512u * U);
    return r.n_pages * (u64)(spp / cc_scan_group<U>(r, nwarps));
}

template <int U>
__device__ __forceinline__ void cc_scan_items(const cc_region_dev& r, u64 first, u64 step) {
    const u32 lane = threadIdx.x & 31u;
    constexpr u32 SEGV = 32u * U;            // vectors per segment
    constexpr u32 SEGB = SEGV * 16u;         // bytes per segment
    const u32 P = r.page_bytes;
    const u32 spp = (P + SEGB - 1) / SEGB;
    const bool pow2 = (spp & (spp - 1)) == 0;
    const bool uniform = (r.bytes % P == 0) && (P % SEGB == 0);
    const u32 G = cc_scan_group<U>(r, step);
    const u32 cpp = spp / G;                 // items per page (G divides spp: both powers of two, or G == 1)
    const u32 csh = 31 - __clz(cpp);
    const u64 n_items = r.n_pages * (u64)cpp;
    for (u64 item = first; item < n_items; item += step) {
        u64 p;
        u32 ch;
        if (pow2) { p = item >> csh; ch = (u32)(item & (cpp - 1)); }
        else { p = item / cpp; ch = (u32)(item - p * cpp); }
        bool dirty = false;
        for (u32 c = 0; c < G && !dirty; c++) {
            const u32 s = ch * G + c;
            const u64 start = p * (u64)P + (u64)s * SEGB;
            const uint4* a = reinterpret_cast<const uint4*>(r.base + start);
            const uint4* b = reinterpret_cast<const uint4*>(r.shadow + start);
            u32 acc = 0;
            if (uniform) {
                uint4 va[U], vb[U];
#pragma unroll
                for (int u = 0; u < U; u++) va[u] = ld_stream(a + lane + 32 * u);
#pragma unroll
                for (int u = 0; u < U; u++) vb[u] = ld_stream(b + lane + 32 * u);
#pragma unroll
                for (int u = 0; u < U; u++)
                    acc |= (va[u].x ^ vb[u].x) | (va[u].y ^ vb[u].y) | (va[u].z ^ vb[u].z) | (va[u].w ^ vb[u].w);
            } else {
                const u64 plen = page_len_dev(r, p);
                const u64 so = (u64)s * SEGB;
                if (so >= plen) break;
                const u64 rem = plen - so;
                const u32 nv = (u32)((rem < SEGB ? rem : SEGB) >> 4);
#pragma unroll
                for (int u = 0; u < U; u++) {
                    const u32 j = lane + 32 * u;
                    if (j < nv) {
                        uint4 x = ld_stream(a + j), y = ld_stream(b + j);
                        acc |= (x.x ^ y.x) | (x.y ^ y.y) | (x.z ^ y.z) | (x.w ^ y.w);
                    }
                }
            }
            dirty = __any_sync(0xFFFFFFFFu, acc != 0);
        }
        if (dirty && lane == 0) atomicOr(&r.bitmap[p >> 5], 1u << (p & 31));
    }
}

template <int U>
__device__ __forceinline__ void cc_scan_phase(const cc_region_dev& r, cc_grid g) {
    if (g.block == 0 && threadIdx.x == 0) {
        r.hdr->t_start_ns = globaltimer_ns();
        r.hdr->ticket = 0;
        r.hdr->run_id = r.hdr->run_id + 1;
    }
    cc_scan_items<U>(r, g.warp(), g.nwarps());
}

// ------------------------------------------------------------------ a2: compaction --
// Ascending list D[0..k) of set bits of the bitmap and k ("dirty page
// descriptors").  Single pass: tiles of 1024 bitmap words are handed out by ticket (so a tile's
// predecessors have always started), each tile publishes its popcount and resolves its exclusive
// prefix by decoupled look-back over run-tagged status words.  The bitmap words are cleared as
// they are consumed.  The block that owns the last tile also writes the plan of the gather:
// record count, byte need, log-full decision (all-or-nothing, reading #10).
#define CC_LB_AGG 1ull
#define CC_LB_INC 2ull
__device__ __forceinline__ u64 lb_pack(u32 run, u64 flag, u32 val) { return ((u64)run << 34) | (flag << 32) | val; }

#define CC_MODE_CHECKPOINT 0u
#define CC_MODE_SCAN_ONLY 1u

// The plan of the record writer, written once k is final (one thread): record count, byte need,
// all-or-nothing log-full decision (reading #10), start offset.  last_dirty: the region's (possibly
// short) last page is among the k pages.  inline_done: the records are already in place (fused pass).
__device__ __forceinline__ void cc_plan_checkpoint_at(const cc_region_dev& r, const cc_log_dev* log, u64 W, u32 mode, u64 epoch,
                                                      u32 k, bool last_dirty, bool inline_done) {
    cc_ws_hdr* h = r.hdr;
    h->k = k;
    h->epoch = epoch;
    u64 need = (u64)k * (CC_RECORD_HEADER_BYTES + (u64)r.page_bytes) + CC_COMMIT_RECORD_BYTES;
    if (last_dirty) need -= (u64)r.page_bytes - page_len_dev(r, r.n_pages - 1);
    int32_t st = CC_OK;
    u32 k_eff = 0;
    if (mode == CC_MODE_CHECKPOINT && k != 0) {
        if (log->buf == nullptr || W + need > log->capacity) st = CC_ERR_LOG_FULL;
        else k_eff = k;
    }
    h->k_eff = k_eff;
    h->commit_k = k_eff;
    h->status = st;
    h->W_start = W;
    h->need = k_eff ? need : 0;
    h->gather_done = 0;
    h->inline_done = inline_done ? 1u : 0u;
}
__device__ __forceinline__ void cc_plan_checkpoint(const cc_region_dev& r, const cc_log_dev* log, u32 mode, u64 epoch, u32 k,
                                                   bool last_dirty, bool inline_done) {
    cc_plan_checkpoint_at(r, log, log->W, mode, epoch, k, last_dirty, inline_done);
}

// Only the first CC_COMPACT_THREADS threads of a block work (the worker's blocks may be wider);
// every thread takes part in the barriers.
__device__ __forceinline__ void cc_compact_phase(const cc_region_dev& r, const cc_log_dev* log, u32 mode, u64 epoch,
                                                 cc_result* out) {
    __shared__ u32 s_ticket, s_excl, s_last_dirty;
    __shared__ u32 s_warp[CC_COMPACT_THREADS / 32];
    const u32 tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5;
    const u32 run = r.hdr->run_id & 0x3FFFFFFFu;
    const u32 nt = (u32)((r.n_words + CC_COMPACT_TILE_WORDS - 1) / CC_COMPACT_TILE_WORDS);
    const u32 nwarp = CC_COMPACT_THREADS / 32;
    const bool active = tid < CC_COMPACT_THREADS;
    for (;;) {
        if (tid == 0) { s_ticket = atomicAdd(&r.hdr->ticket, 1u); s_last_dirty = 0; }
        __syncthreads();
        const u32 t = s_ticket;
        if (t >= nt) break;
        // each thread owns CC_COMPACT_WORDS_PER_THREAD consecutive words per 'row' of blockDim threads
        u32 cnt = 0;
        constexpr u32 words_per_thread = CC_COMPACT_WORDS_PER_THREAD;
        const u64 w0 = (u64)t * CC_COMPACT_TILE_WORDS + (u64)tid * words_per_thread;
        u32 wv[words_per_thread] = {0, 0, 0, 0};
        if (active) {
            uint4 q = *reinterpret_cast<const uint4*>(&r.bitmap[w0]);   // bitmap is padded to whole tiles
            wv[0] = q.x; wv[1] = q.y; wv[2] = q.z; wv[3] = q.w;
            if (q.x | q.y | q.z | q.w) *reinterpret_cast<uint4*>(&r.bitmap[w0]) = make_uint4(0, 0, 0, 0);
            cnt = __popc(q.x) + __popc(q.y) + __popc(q.z) + __popc(q.w);
        }
        // block exclusive scan of cnt
        u32 inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 n = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= o) inc += n;
        }
        if (lane == 31 && active) s_warp[wid] = inc;
        __syncthreads();
        u32 warp_base = 0, total = 0;
        for (u32 i = 0; i < nwarp; i++) {
            u32 v = s_warp[i];
            if (i < wid) warp_base += v;
            total += v;
        }
        if (tid == 0) {
            u32 excl = 0;
            if (t == 0) {
                st_release_gpu_u64(&r.lb_status[0], lb_pack(run, CC_LB_INC, total));
            } else {
                st_release_gpu_u64(&r.lb_status[t], lb_pack(run, CC_LB_AGG, total));
                int j = (int)t - 1;
                while (j >= 0) {
                    u64 s = ld_acquire_gpu_u64(&r.lb_status[j]);
                    if ((u32)(s >> 34) != run || ((s >> 32) & 3ull) == 0) { __nanosleep(20); continue; }
                    excl += (u32)s;
                    if (((s >> 32) & 3ull) == CC_LB_INC) break;
                    j--;
                }
                st_release_gpu_u64(&r.lb_status[t], lb_pack(run, CC_LB_INC, excl + total));
            }
            s_excl = excl;
        }
        __syncthreads();
        u32 pos = s_excl + warp_base + (inc - cnt);
#pragma unroll
        for (u32 i = 0; i < words_per_thread; i++) {
            u32 w = wv[i];
            const u64 pbase = (w0 + i) << 5;
            while (w) {
                const u32 bit = __ffs(w) - 1;
                w &= w - 1;
                const u64 page = pbase + bit;
                r.D[pos++] = (u32)page;
                if (page == r.n_pages - 1) s_last_dirty = 1;
            }
        }
        __syncthreads();
        if (t == nt - 1 && tid == 0) {
            const u32 k = s_excl + total;
            cc_ws_hdr* h = r.hdr;
            cc_plan_checkpoint(r, log, mode, epoch, k, s_last_dirty != 0, false);
            const u64 W = h->W_start;
            if (mode == CC_MODE_SCAN_ONLY && out) {
                out->n_dirty = k;
                out->bytes = 0;
                out->log_offset_after = W;
                out->epoch = epoch;
                out->status = CC_OK;
                out->flags = CC_TASK_NOP;
                out->t_start_ns = h->t_start_ns;
                out->t_end_ns = globaltimer_ns();
                __threadfence_system();
                st_release_sys_u64(&out->seq_done, 1ull);
            }
            __threadfence();
        }
        __syncthreads();
    }
}

// Base snapshot ("The initial base snapshot captured all 8,192 pages"):
// every page is a record -- D = 0..n_pages-1, no discovery at all; the gather below does the rest.
__device__ __forceinline__ void cc_snapshot_plan_phase(const cc_region_dev& r, const cc_log_dev* log, u64 epoch, cc_grid g) {
    for (u64 i = (u64)g.block * blockDim.x + threadIdx.x; i < r.n_pages; i += (u64)g.nblocks * blockDim.x) r.D[i] = (u32)i;
    if (g.block == 0 && threadIdx.x == 0) {
        r.hdr->t_start_ns = globaltimer_ns();
        cc_plan_checkpoint(r, log, CC_MODE_CHECKPOINT, epoch, (u32)r.n_pages, true, false);
    }
}

#ifndef CC_GATHER_CHUNK_LOG2
#define CC_GATHER_CHUNK_LOG2 2u
#endif
#define CC_GATHER_CHUNK (1u << CC_GATHER_CHUNK_LOG2)      // consecutive 4 KiB segments of a record one warp takes at a time (cc_gather_items)

// ------------------------------------------------- a3-a5: gather + CRC + commit + shadow --
// For record i < k_eff: header {region_id, D[i], len, crc32c(payload)} + payload at
// W_start + i*(16+P), and shadow[page] := cur[page] (L264).  One warp moves
// one 4 KiB segment: the bytes are read ONCE into registers and the log payload, the shadow and
// the CRC all come from that one read.  The warp that completes a record's last segment writes
// its header.  Every block fences its stores at system scope and counts itself done; the last
// block appends the commit record, fences, publishes the committed offset with a system-scope
// release store (L263: "a commit marker publishes the epoch only after all bytes are visible")
// and fills the result.
__device__ __forceinline__ void st_u32x4(u8* p, u32 a, u32 b, u32 c, u32 d) {
    uint4 v = make_uint4(a, b, c, d);
    st_stream(reinterpret_cast<uint4*>(p), v);
}

// One (record, segment) item of the record writer: segment c of page p, which is record i of the checkpoint that starts
// at log offset W0.  The warp reads the segment ONCE; log payload, shadow and CRC contribution come from that read.
// Returns the segment's CRC contribution (in every lane); 0 for a segment beyond the page's end.
__device__ __forceinline__ u32 cc_gather_segment_copy(const cc_region_dev& r, cc_dev* dev, cc_crc_smem* cs, u64 W0, u32 i, u32 c, u32 p,
                                                      u32 lane) {
    constexpr int U = 8;
    cc_log_dev* log = &dev->log;
    const u32 P = r.page_bytes;
    const u64 plen = page_len_dev(r, p);
    const u64 so = (u64)c * CC_SEG_BYTES;
    if (so >= plen) return 0u;
    const u64 rem = plen - so;
    const u32 seg_len = (u32)(rem < CC_SEG_BYTES ? rem : CC_SEG_BYTES);
    const u32 nv = seg_len >> 4;
    const u64 after = rem - seg_len;
    const u64 src_off = (u64)p * P + so;
    const uint4* src = reinterpret_cast<const uint4*>(r.base + src_off);
    const bool has_shadow = r.shadow != nullptr;      // allocator-aware regions may have none (cc_mark.cuh)
    uint4* dsh = reinterpret_cast<uint4*>(r.shadow + src_off);
    u8* rec = log->buf + W0 + (u64)i * ((u64)P + CC_RECORD_HEADER_BYTES);
    uint4* dlog = reinterpret_cast<uint4*>(rec + CC_RECORD_HEADER_BYTES + so);
    uint4 v[U];
    if (nv == CC_SEG_VECS) {
#pragma unroll
        for (int u = 0; u < U; u++) v[u] = ld_stream(src + lane + 32 * u);
#pragma unroll
        for (int u = 0; u < U; u++) st_stream(dlog + lane + 32 * u, v[u]);
        if (has_shadow) {
#pragma unroll
            for (int u = 0; u < U; u++) st_stream(dsh + lane + 32 * u, v[u]);
        }
    } else {
#pragma unroll
        for (int u = 0; u < U; u++) {
            const u32 j = lane + 32 * u;
            if (j < nv) {
                v[u] = ld_stream(src + j);
                st_stream(dlog + j, v[u]);
                if (has_shadow) st_stream(dsh + j, v[u]);
            } else {
                v[u] = make_uint4(0, 0, 0, 0);
            }
        }
    }
    return crc_segment_warp<U>(cs, &dev->crc, v, nv, after, lane);
}

// Segments c0 .. c0 + cn - 1 of record i are in place (contrib = XOR of their contributions; segments beyond the page's
// end count as done): the warp that completes the record writes its header.
__device__ __forceinline__ void cc_gather_record_done(const cc_region_dev& r, cc_dev* dev, u64 W0, u32 i, u32 p, u32 c0, u32 cn,
                                                      u32 contrib, u32 lane) {
    if (lane != 0) return;
    const u32 P = r.page_bytes;
    const u64 plen = page_len_dev(r, p);
    const u32 nseg = (u32)((plen + CC_SEG_BYTES - 1) / CC_SEG_BYTES);
    if (c0 >= nseg) return;
    if (c0 + cn > nseg) cn = nseg - c0;
    u32 acc = 0;
    if (crc_record_combine_n(&r.rec_state[i], nseg, c0, cn, contrib, &acc)) {
        u8* rec = dev->log.buf + W0 + (u64)i * ((u64)P + CC_RECORD_HEADER_BYTES);
        st_u32x4(rec, r.region_id, p, (u32)plen, crc_finalize(acc, plen == P ? r.crc_init_full : r.crc_init_tail));
    }
}

__device__ __forceinline__ void cc_gather_segment(const cc_region_dev& r, cc_dev* dev, cc_crc_smem* cs, u64 W0, u32 i, u32 c, u32 p,
                                                  u32 lane) {
    const u32 contrib = cc_gather_segment_copy(r, dev, cs, W0, i, c, p, lane);
    cc_gather_record_done(r, dev, W0, i, p, c, 1u, contrib, lane);
}

// The record writer proper (no synchronisation with other blocks): items first, first + step, ... of the
// region's k_eff * spp (record, segment) items.  cs must hold the CRC tables.
__device__ __forceinline__ void cc_gather_items(const cc_region_dev& r, cc_dev* dev, cc_crc_smem* cs, u64 first, u64 step) {
    cc_ws_hdr* h = r.hdr;
    const u32 k_eff = h->k_eff;
    const u32 lane = threadIdx.x & 31u;
    const u64 W0 = h->W_start;
    const u32 spp = r.spp;
    const u64 n_items = (u64)k_eff * spp;
    // A warp takes CC_GATHER_CHUNK consecutive segments of one record at a time when pages have that many and there are
    // chunks enough to go round (>= 4 per warp): one look at D[], one 64-bit atomic on the record's state word per chunk
    // instead of per segment.  Item numbering (first, first + step, ...) then counts chunks.
    u32 G = 1;
    if (r.spp_shift >= (int)CC_GATHER_CHUNK_LOG2 && n_items / CC_GATHER_CHUNK >= 4 * step) G = CC_GATHER_CHUNK;
    if (G == 1) {
        for (u64 item = first; item < n_items; item += step) {
            u32 i, c;
            if (r.spp_shift >= 0) { i = (u32)(item >> r.spp_shift); c = (u32)(item & (spp - 1)); }
            else { i = (u32)(item / spp); c = (u32)(item - (u64)i * spp); }
            cc_gather_segment(r, dev, cs, W0, i, c, r.D[i], lane);
        }
        return;
    }
    const u64 n_chunks = n_items / G;                          // spp is a power of two >= G: whole chunks
    const u32 cps_shift = (u32)r.spp_shift - CC_GATHER_CHUNK_LOG2;      // log2(chunks per page)
    for (u64 ch = first; ch < n_chunks; ch += step) {
        const u32 i = (u32)(ch >> cps_shift);
        const u32 c0 = (u32)(ch & ((1u << cps_shift) - 1u)) * G;
        const u32 p = r.D[i];
        u32 contrib = 0;
#pragma unroll 1
        for (u32 q = 0; q < G; q++) contrib ^= cc_gather_segment_copy(r, dev, cs, W0, i, c0 + q, p, lane);
        cc_gather_record_done(r, dev, W0, i, p, c0, G, contrib, lane);
    }
}

__device__ __forceinline__ void cc_gather_work(const cc_region_dev& r, cc_dev* dev, cc_crc_smem* cs, cc_grid g, bool init_tables) {
    const cc_ws_hdr* h = r.hdr;
    const u32 k_eff = h->k_eff;
    // warps take items round-robin, so a block has work iff its first warp index is < n_items
    // (after a fused pass that already wrote the records -- cc_fused.cuh -- only the commit is left)
    if (k_eff != 0 && !h->inline_done && (u64)g.block * (blockDim.x >> 5) < (u64)k_eff * r.spp) {
        if (init_tables) cc_crc_smem_init(cs, &dev->crc);
        if (g.block == 0 && threadIdx.x == 0) CC_TRACE(dev, 5);
        cc_gather_items(r, dev, cs, g.warp(), g.nwarps());
        if (g.block == 0 && threadIdx.x == 0) CC_TRACE(dev, 9);
    }
}

// One thread: the region's commit record ("write commit marker"); returns the offset after it
// (W_start if nothing was appended).  Also re-arms the per-region counters for the next call.
__device__ __forceinline__ u64 cc_gather_commit_record(const cc_region_dev& r, cc_dev* dev) {
    cc_ws_hdr* h = r.hdr;
    cc_log_dev* log = &dev->log;
    const u32 k_eff = h->k_eff;
    const u64 W0 = h->W_start;
    u64 W_after = W0;
    if (k_eff != 0) {
        u8* c = log->buf + W0 + h->need - CC_COMMIT_RECORD_BYTES;
        const u64 epoch = h->epoch;
        u32 pay[4] = {(u32)epoch, (u32)(epoch >> 32), r.region_id, h->commit_k};
        const u32 crc = crc_serial(&dev->crc, reinterpret_cast<const u8*>(pay), 16);
        st_u32x4(c + 16, pay[0], pay[1], pay[2], pay[3]);
        st_u32x4(c, CC_COMMIT_ID, CC_COMMIT_ID, 16u, crc);
        W_after = W0 + h->need;
    }
    h->gather_done = 0;
    h->fticket = 0;
    h->frun = h->frun + 1;
    return W_after;
}

// Completion of a region's record writer.  Every block that wrote records orders its stores before one gpu-scope
// atomic on the region's counter (bar.sync, then ONE thread: fence.gpu + atomicAdd -- the fence is cumulative over what
// the barrier ordered before it); the block that counts last has, by that chain, every block's record bytes behind it:
// it appends the commit record, fills the result, executes the ONE system-scope fence of the call and only then stores
// the publishing words (L263 "a commit marker publishes the epoch only after all bytes are visible").  System-scope
// fences cost microseconds each (more with host-link stores in flight); a chain of four of them per call -- every
// thread, then one thread per block, then two in the last block -- was 15-20 us of a 55 us checkpoint of a 64 MiB region.
// Only the blocks that had items take part (n_items = items of the record writer; at least block 0): with a
// small dirty set the other blocks leave at once instead of queueing atomics on one counter.
__device__ __forceinline__ void cc_gather_complete(const cc_region_dev& r, cc_dev* dev, cc_grid g, cc_result* out, u32 kind,
                                                   u64 n_items) {
    cc_ws_hdr* h = r.hdr;
    cc_log_dev* log = &dev->log;
    const u64 wpb = blockDim.x >> 5;
    u64 n_work = (n_items + wpb - 1) / wpb;
    if (n_work > g.nblocks) n_work = g.nblocks;
    if (n_work == 0) n_work = 1;
    if (g.block >= n_work) return;
    __shared__ u32 s_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = (atomicAdd(&h->gather_done, 1u) == (u32)n_work - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        CC_TRACE(dev, 6);
        __threadfence();                        // (acquire side of the counter: every block's record bytes are behind us)
        const bool appended = h->k_eff != 0;
        const u64 W_after = cc_gather_commit_record(r, dev);
        CC_TRACE(dev, 7);
        if (out) {
            out->n_dirty = h->k;
            out->bytes = h->need;
            out->log_offset_after = W_after;
            out->epoch = h->epoch;
            out->status = h->status;
            out->flags = kind;
            out->t_start_ns = h->t_start_ns;
            out->t_end_ns = globaltimer_ns();
        }
        // ONE system-scope fence behind the record bytes (all blocks'), the commit record and the result fields, then
        // the publishing words
        __threadfence_system();
        if (appended) cc_log_publish_fenced(log, W_after);
        if (out) st_relaxed_sys_u64(&out->seq_done, 1ull);
        CC_TRACE(dev, 8);
    }
}

__device__ __forceinline__ void cc_gather_phase(const cc_region_dev& r, cc_dev* dev, cc_crc_smem* cs, cc_grid g,
                                                cc_result* out, u32 kind, bool init_tables) {
    const u64 n_items = r.hdr->inline_done ? 0ull : (u64)r.hdr->k_eff * r.spp;
    cc_gather_work(r, dev, cs, g, init_tables);
    cc_gather_complete(r, dev, g, out, kind, n_items);
}
