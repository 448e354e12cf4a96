// cc_pass.cuh -- the single-pass checkpoint: discovery (a1) + ordered ranking (a2) + record writer with CRC32C (a3) +
// shadow update (a5) + commit and publish (a4) in ONE kernel, with no block-level synchronisation on its fast path
// (SURVEY.md 8f #2 "scan -> offset (decoupled look-back) -> gather in one kernel").
//
// The unit of work is a WARP TILE of 1..32 consecutive pages, handed out by ticket.  A warp
//   discovers   its tile's dirty mask (one register): compare live vs shadow page by page, stopping a page at its
//               first differing 4 KiB segment (early-out) -- or takes it from the runtime's dirty bitmap / version
//               counters (allocator-aware discovery), or "all pages" (base snapshot, L394);
//   ranks       it: the tile's page count (and, for run-length records, its record count) is published and the sums
//               over all earlier tiles are resolved by a warp-wide decoupled look-back (32 predecessors per step), so
//               the dirty list comes out ascending and every record knows its final log offset
//               W + 16 * (records before) + P * (pages before);
//   writes      its own records right away: one read of a segment feeds the log payload, the shadow and the CRC32C
//               (a running Horner product over the record's segments, in a register); a record is one page, or --
//               PAPER.md:L221 "contiguous dirty ranges use run-length encoding" -- one RUN of consecutive dirty pages.
//               Runs are cut at tile boundaries, and tiles are whole multiples of run_pages, so no run crosses a tile
//               and the bytes are exactly those of the oracle's run records;
//   leaves      every warp counts itself out (per block in shared memory, then one gpu-scope atomic per block); the
//               LAST warp of the grid appends the commit record, fills the result, executes the call's one
//               system-scope fence and publishes the committed offset (L263).
// All-or-nothing (reading #10) is decided up front: records are written inline only if the WORST case (every page
// dirty) fits behind the write offset.  Otherwise the same kernel falls back to the classic phases (scan, compaction,
// [run ranking,] gather) separated by grid barriers -- which is why it is launched cooperatively.
#pragma once
#include "cc_common.cuh"
#include "cc_crc.cuh"
#include "cc_ckpt.cuh"
#include "cc_mark.cuh"
#include "cc_rle.cuh"
#include "cc_fused.cuh"

// cc_pass_args.disc: CC_DISC_SCAN / _MARKS / _VERSIONS / _ALL of concordia.h, and internally
#define CC_DISC_MARKS_VERIFY 2u     // the runtime's bitmap narrows the compare (CC_DISC_MARKS + CC_MARK_VERIFY)

#define CC_PASS_MAX_TILES (1u << 20)

struct cc_pass_args {
    u64 epoch;
    u32 disc;               // CC_DISC_*
    u32 run_pages;          // <= 1: one record per page; 2..32: run-length records
    u32* marks;             // CC_DISC_MARKS*: the caller's bitmap
    u32 consume;            // ... cleared after a successful checkpoint
    u32 kind;               // task kind echoed into the result
    const u64* version;     // CC_DISC_VERSIONS
    u64* committed;
};

// Pages per warp tile for this call: about one tile per warp of the grid for small regions (every tile costs one atomic
// on the ticket counter), at most ~32 KiB of region per tile (a warp that finds a dirty page waits for its
// predecessors: a 256 MiB / 4 KiB-page task took 179 us with 64 KiB tiles and 116 us with 16-32 KiB tiles), at most
// CC_PASS_MAX_TILES tiles, and a whole multiple of run_pages.  (profiles/r02_pass_probe.md: 8 / 16 / 32 / 64 KiB tiles.)
__device__ __forceinline__ u32 cc_pass_tile_pages(const cc_region_dev& r, u32 run_pages, u32 nwarps) {
    const u64 n = r.n_pages;
    u64 tp = (n + nwarps - 1) / nwarps;
    const u64 cap = CC_FUSED_TILE_BYTES / r.page_bytes;
    if (tp > cap) tp = cap;
    const u64 lo = (n + CC_PASS_MAX_TILES - 1) / CC_PASS_MAX_TILES;
    if (tp < lo) tp = lo;
    if (tp < 1) tp = 1;
    if (tp > 32) tp = 32;
    if (run_pages > 1) {
        u64 t = tp / run_pages * run_pages;
        if (t < run_pages) t = run_pages;
        // rounding down must not undo the lower bound: more than CC_PASS_MAX_TILES tiles would run past the look-back
        // words the workspace holds.  Rounding `lo` UP stays <= 32 for every shape cc_pass_supported admits.
        if (t < lo) t = (lo + run_pages - 1) / run_pages * run_pages;
        tp = t;
    }
    return (u32)tp;
}
// The single pass takes a region iff it can be cut into at most CC_PASS_MAX_TILES tiles: a tile has at most 32 pages
// (one mask register) and is a whole multiple of run_pages, so at most 32 / run_pages * run_pages pages.
__host__ __device__ __forceinline__ bool cc_pass_supported(u64 n_pages, u32 run_pages) {
    if (run_pages > 32) return false;
    const u64 tmax = run_pages > 1 ? 32u / run_pages * run_pages : 32u;
    return n_pages <= tmax * CC_PASS_MAX_TILES;
}

// Shared-memory CRC tables, filled on first use by the warp that needs them (most blocks of a sparse checkpoint
// never do): state 0 = empty, 1 = being filled, 2 = ready.
__device__ __forceinline__ void cc_crc_smem_lazy(cc_crc_smem* s, const cc_crc_tables* g, u32* state, u32 lane) {
    u32 st = *reinterpret_cast<volatile u32*>(state);
    if (st == 2u) return;
    if (lane == 0) st = atomicCAS(state, 0u, 1u);
    st = __shfl_sync(0xFFFFFFFFu, st, 0);
    if (st == 0u) {                                           // this warp fills them
        for (u32 e0 = 0; e0 < 256u; e0 += 32u) {
            const u32 mine = rotl32(g->t0[e0 + lane], 7);
#pragma unroll
            for (u32 e = 0; e < 32u; e++) s->t0[(e0 + e) * 32u + lane] = __shfl_sync(0xFFFFFFFFu, mine, e);
        }
        const uint4* nib = reinterpret_cast<const uint4*>(g->lane_nib);
        uint4* dn = reinterpret_cast<uint4*>(s->lane_nib);
        for (u32 i = lane; i < 8 * 16 * 32 / 4; i += 32) dn[i] = nib[i];
        const uint4* s5 = reinterpret_cast<const uint4*>(&g->s512[0][0]);
        uint4* d5 = reinterpret_cast<uint4*>(s->s512);
        for (u32 i = lane; i < 4 * 256 / 4; i += 32) d5[i] = s5[i];
        __syncwarp();
        __threadfence_block();
        if (lane == 0) atomicExch(state, 2u);
    } else {
        while (*reinterpret_cast<volatile u32*>(state) != 2u) __nanosleep(50);
    }
    __threadfence_block();
}

// compare one page with its shadow, stop at the first differing segment
__device__ __forceinline__ bool cc_pass_page_dirty(const cc_region_dev& r, u64 p, u32 lane) {
    constexpr int U = 8;
    const u32 P = r.page_bytes;
    const u64 plen = page_len_dev(r, p);
    const uint4* a = reinterpret_cast<const uint4*>(r.base + p * (u64)P);
    const uint4* b = reinterpret_cast<const uint4*>(r.shadow + p * (u64)P);
    const u32 nvec = (u32)(plen >> 4);
    bool dirty = false;
    for (u32 v0 = 0; v0 < nvec && !dirty; v0 += CC_SEG_VECS) {
        u32 acc = 0;
        if (v0 + CC_SEG_VECS <= nvec) {
            uint4 va[U], vb[U];
#pragma unroll
            for (int u = 0; u < U; u++) va[u] = ld_stream(a + v0 + lane + 32 * u);
#pragma unroll
            for (int u = 0; u < U; u++) vb[u] = ld_stream(b + v0 + lane + 32 * u);
#pragma unroll
            for (int u = 0; u < U; u++)
                acc |= (va[u].x ^ vb[u].x) | (va[u].y ^ vb[u].y) | (va[u].z ^ vb[u].z) | (va[u].w ^ vb[u].w);
        } else {
#pragma unroll
            for (int u = 0; u < U; u++) {
                const u32 j = v0 + lane + 32 * u;
                if (j < nvec) {
                    uint4 x = ld_stream(a + j), y = ld_stream(b + j);
                    acc |= (x.x ^ y.x) | (x.y ^ y.y) | (x.z ^ y.z) | (x.w ^ y.w);
                }
            }
        }
        dirty = __any_sync(0xFFFFFFFFu, acc != 0);
    }
    return dirty;
}

// Completion of a single-pass call: every warp of the grid comes here once.  s_warps_left: shared counter of the
// block, preset to its warp count.  Returns true in the ONE warp of the grid that leaves last.  No system-scope fence
// here: a warp orders its record / shadow stores before its count-out at block scope, the block's last warp before the
// grid counter at gpu scope, and the grid's last warp executes the call's one system-scope fence behind the commit
// record (cc_pass_commit) -- fences are cumulative along that chain.
__device__ __forceinline__ bool cc_pass_leave(cc_ws_hdr* h, u32* s_warps_left, bool wrote, u32 nblocks, u32 lane) {
    __syncwarp();
    u32 last = 0;
    if (lane == 0) {
        if (wrote) __threadfence_block();
        if (atomicSub(s_warps_left, 1u) == 1u) {              // last warp of the block
            __threadfence();
            last = (atomicAdd(&h->gather_done, 1u) == nblocks - 1) ? 1u : 0u;
            if (last) __threadfence();
        }
    }
    return __shfl_sync(0xFFFFFFFFu, last, 0) != 0;
}

// CC_MARK_CONSUME: clear the tile's bits of the caller's bitmap (the tile may straddle two words); the region's last
// tile also clears the last word's bits beyond n_pages (the whole bitmap ends up zero).
__device__ __forceinline__ void cc_pass_clear_marks(const cc_region_dev& r, const cc_pass_args& a, u64 p0, u32 np, bool last_tile) {
    const u32 tile_bits = np == 32 ? 0xFFFFFFFFu : ((1u << np) - 1u);
    const u64 wi = p0 >> 5;
    const u32 sh = (u32)(p0 & 31u);
    const u64 clr = (u64)tile_bits << sh;
    const u32 lo = (u32)clr, hi = (u32)(clr >> 32);
    if (lo && (a.marks[wi] & lo)) atomicAnd(&a.marks[wi], ~lo);
    if (hi && wi + 1 < r.n_words && (a.marks[wi + 1] & hi)) atomicAnd(&a.marks[wi + 1], ~hi);
    if (last_tile) {
        const u32 valid = (u32)(((r.n_pages - 1) & 31u) + 1u);
        if (valid < 32) {
            const u32 junk = ~((1u << valid) - 1u);
            if (a.marks[r.n_words - 1] & junk) atomicAnd(&a.marks[r.n_words - 1], ~junk);
        }
    }
}

// The inline single pass over the tiles (see the file header).  Whole warps call this; no block barrier inside.
// Tiles are handed out by an atomic TICKET, so that a tile's predecessors have always started -- and, being taken in
// time order, have mostly FINISHED: the look-back then finds an inclusive sum within a step or two.  A ticket is drawn
// only when the warp is ready for the tile: drawing the next one ahead of time (to hide the atomic's latency) hands out
// every tile in the first microseconds -- a static deal in disguise, in which a dirty tile waits on predecessors that
// sit in some other warp's queue (profiles/r02_pass_probe.md: a 256 MiB ring task took 156 us instead of 109 us, an
// 8 GiB checkpoint into a pinned log 16.2 ms instead of 12.0 ms).
// Returns whether this warp stored record or shadow bytes.
__device__ __forceinline__ bool cc_pass_tiles(const cc_region_dev& r, cc_dev* dev, cc_crc_smem* cs, u32* s_crc_state,
                                              const cc_pass_args& a, u32 TP, u64 W0, cc_grid) {
    constexpr int U = 8;
    cc_ws_hdr* h = r.hdr;
    cc_log_dev* log = &dev->log;
    const u32 lane = threadIdx.x & 31u;
    const u32 P = r.page_bytes;
    const u32 nt = (u32)((r.n_pages + TP - 1) / TP);
    const u32 run = h->frun & 0x3FFFFFFFu;
    const bool rle = a.run_pages > 1;
    const bool has_shadow = r.shadow != nullptr;
    const u32 pow_lane = dev->crc.seg_pow[32 + lane];
    // bits of a tile at multiples of run_pages (tiles start at multiples of run_pages)
    u32 cut = 0xFFFFFFFFu;
    if (rle) { cut = 0; for (u32 q = 0; q < 32; q += a.run_pages) cut |= 1u << q; }
    bool wrote = false;
    for (;;) {
        u32 t = 0;
        if (lane == 0) t = atomicAdd(&h->fticket, 1u);
        t = __shfl_sync(0xFFFFFFFFu, t, 0);
        if (t >= nt) break;
        const u64 p0 = (u64)t * TP;
        const u32 np = (u32)((r.n_pages - p0) < TP ? (r.n_pages - p0) : TP);
        const u32 tile_bits = np == 32 ? 0xFFFFFFFFu : ((1u << np) - 1u);
        // ---- a1: the tile's dirty mask ----
        u32 mask = 0;
        if (a.disc == CC_DISC_ALL) mask = tile_bits;
        else if (a.disc == CC_DISC_VERSIONS) {
            const bool d = lane < np && a.version[p0 + lane] != a.committed[p0 + lane];
            mask = __ballot_sync(0xFFFFFFFFu, d);
        } else {
            if (a.disc != CC_DISC_SCAN) {                     // the runtime's marks: the tile may straddle two words
                const u64 wi = p0 >> 5;
                u64 bits = a.marks[wi];
                if (wi + 1 < r.n_words) bits |= (u64)a.marks[wi + 1] << 32;
                mask = (u32)(bits >> (p0 & 31u)) & tile_bits;
            }
            if (a.disc != CC_DISC_MARKS) {
                u32 todo = a.disc == CC_DISC_SCAN ? tile_bits : mask;
                mask = 0;
                while (todo) {
                    const u32 pl = (u32)__ffs(todo) - 1u;
                    todo &= todo - 1;
                    if (cc_pass_page_dirty(r, p0 + pl, lane)) mask |= 1u << pl;
                }
            }
        }
        // ---- a2: rank of this tile's dirty pages (and records) among all ----
        const u32 cnt = __popc(mask);
        CC_TRACE_MAX(dev, cnt ? 20 : 23, lane);
        const u32 starts = rle ? (mask & (~(mask << 1) | cut)) : mask;
        const u32 nrec = __popc(starts);
        const bool last = (t == nt - 1);
        u32 excl = 0, excl_r = 0;
        if (cnt == 0 && !last) {
            // nothing to place: publish, upgrading to an inclusive sum only if that costs no waiting
            const bool got = cc_fused_lookback(r.flb_status, run, t, lane, false, &excl, 2);
            if (lane == 0) st_relaxed_gpu_u64(&r.flb_status[t], got ? lb_pack(run, CC_LB_INC, excl) : lb_pack(run, CC_LB_AGG, 0));
            if (rle) {
                const bool got2 = cc_fused_lookback(r.lb2, run, t, lane, false, &excl_r, 2);
                if (lane == 0) st_relaxed_gpu_u64(&r.lb2[t], got2 ? lb_pack(run, CC_LB_INC, excl_r) : lb_pack(run, CC_LB_AGG, 0));
            }
        } else {
            if (t != 0 && lane == 0) {
                st_relaxed_gpu_u64(&r.flb_status[t], lb_pack(run, CC_LB_AGG, cnt));
                if (rle) st_relaxed_gpu_u64(&r.lb2[t], lb_pack(run, CC_LB_AGG, nrec));
            }
            cc_fused_lookback(r.flb_status, run, t, lane, true, &excl);
            if (lane == 0) st_relaxed_gpu_u64(&r.flb_status[t], lb_pack(run, CC_LB_INC, excl + cnt));
            if (rle) {
                cc_fused_lookback(r.lb2, run, t, lane, true, &excl_r);
                if (lane == 0) st_relaxed_gpu_u64(&r.lb2[t], lb_pack(run, CC_LB_INC, excl_r + nrec));
            } else excl_r = excl;
            if ((mask >> lane) & 1u) r.D[excl + __popc(mask & ((1u << lane) - 1u))] = (u32)(p0 + lane);
            if (last && lane == 0) {          // every earlier tile has published its counts: k is final
                const u32 k = excl + cnt, nr = excl_r + nrec;
                u64 need = (u64)nr * CC_RECORD_HEADER_BYTES + (u64)k * P + CC_COMMIT_RECORD_BYTES;
                if ((mask >> (np - 1)) & 1u) need -= (u64)P - page_len_dev(r, r.n_pages - 1);
                h->k = k;
                h->k_eff = k;
                h->commit_k = nr;
                h->n_runs = nr;
                h->epoch = a.epoch;
                h->status = CC_OK;                            // the worst case fits (checked before the pass)
                h->W_start = W0;
                h->need = k ? need : 0;
                h->inline_done = 1;
                // The grid's last warp (cc_pass_commit) reads the plan.  This warp may leave without having written a
                // record (a clean last tile), so cc_pass_leave would not fence for it: order the plan stores before
                // this thread's count-out here, at gpu scope (one warp per call).
                __threadfence();
            }
        }
        // ---- allocator metadata handed back (the checkpoint cannot fail any more: the worst case fits) ----
        if (a.disc == CC_DISC_VERSIONS) {
            if ((mask >> lane) & 1u) a.committed[p0 + lane] = a.version[p0 + lane];
        } else if (a.consume && lane == 0) cc_pass_clear_marks(r, a, p0, np, last);
        if (cnt == 0) continue;
        CC_TRACE_MAX(dev, 21, lane);
        // ---- a3 + a5: this warp writes its own records (one read -> log payload, shadow, CRC) ----
        cc_crc_smem_lazy(cs, &dev->crc, s_crc_state, lane);
        wrote = true;
        u32 m = mask, i = excl_r, rank = excl;
        while (m) {
            const u32 s = (u32)__ffs(m) - 1u;
            // the run that starts at bit s: consecutive set bits up to the next start
            const u32 later_starts = starts & ~((2u << s) - 1u);            // starts above s
            const u32 gap = ~m & ~((1u << s) - 1u);                         // first clear bit at or above s
            u32 end = gap ? (u32)__ffs(gap) - 1u : 32u;
            if (later_starts) { const u32 ns = (u32)__ffs(later_starts) - 1u; if (ns < end) end = ns; }
            const u32 npg = end - s;
            u8* rec = log->buf + W0 + (u64)i * CC_RECORD_HEADER_BYTES + (u64)rank * P;
            u32 crc = 0;
            u64 total = 0;
            for (u32 q = 0; q < npg; q++) {
                const u64 p = p0 + s + q;
                const u64 plen = page_len_dev(r, p);
                const uint4* src = reinterpret_cast<const uint4*>(r.base + p * (u64)P);
                uint4* dsh = reinterpret_cast<uint4*>(r.shadow + p * (u64)P);
                uint4* dlog = reinterpret_cast<uint4*>(rec + CC_RECORD_HEADER_BYTES + total);
                const u32 nvec = (u32)(plen >> 4);
                for (u32 v0 = 0; v0 < nvec; v0 += CC_SEG_VECS) {
                    uint4 v[U];
                    u32 nv = nvec - v0;
                    const bool first = (total == 0 && v0 == 0);
                    if (nv >= CC_SEG_VECS) {
                        nv = CC_SEG_VECS;
#pragma unroll
                        for (int u = 0; u < U; u++) v[u] = ld_stream(src + v0 + lane + 32 * u);
#pragma unroll
                        for (int u = 0; u < U; u++) st_stream(dlog + v0 + lane + 32 * u, v[u]);
                        if (has_shadow) {
#pragma unroll
                            for (int u = 0; u < U; u++) st_stream(dsh + v0 + lane + 32 * u, v[u]);
                        }
                        if (!first) crc = cc_warp_mul_seg(crc, pow_lane, lane);
                    } else {
#pragma unroll
                        for (int u = 0; u < U; u++) {
                            const u32 qv = lane + 32 * u;
                            if (qv < nv) {
                                v[u] = ld_stream(src + v0 + qv);
                                st_stream(dlog + v0 + qv, v[u]);
                                if (has_shadow) st_stream(dsh + v0 + qv, v[u]);
                            } else {
                                v[u] = make_uint4(0, 0, 0, 0);
                            }
                        }
                        if (!first) crc = gf_mul(crc, gf_xpow_bytes(dev->crc.xp, (u64)nv * 16u));
                    }
                    crc ^= crc_segment_warp<U>(cs, &dev->crc, v, nv, 0, lane);
                }
                total += plen;
            }
            if (lane == 0) {
                u32 it;
                if (total == P) it = r.crc_init_full;
                else if (npg == 1) it = r.crc_init_tail;
                else it = gf_mul(0xFFFFFFFFu, gf_xpow_bytes(dev->crc.xp, total));
                st_u32x4(rec, r.region_id, (u32)(p0 + s), (u32)total, crc_finalize(crc, it));
            }
            i++;
            rank += npg;
            m &= ~(((npg == 32 ? 0u : (1u << npg)) - 1u) << s);
        }
        CC_TRACE_MAX(dev, 22, lane);
    }
    return wrote;
}

// The ONE warp that leaves last: commit record, publish, result, and the counters re-armed for the next call.
__device__ __forceinline__ void cc_pass_commit(const cc_region_dev& r, cc_dev* dev, cc_result* out, u32 kind, u32 lane) {
    if (lane != 0) return;
    cc_ws_hdr* h = r.hdr;
    cc_log_dev* log = &dev->log;
    const bool appended = h->k_eff != 0;
    const u64 W_after = cc_gather_commit_record(r, dev);      // (also resets gather_done / fticket, bumps frun)
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
    __threadfence_system();                                   // the call's ONE system-scope fence: behind every warp's records, the commit record and the result
    if (appended) cc_log_publish_fenced(log, W_after);
    if (out) st_relaxed_sys_u64(&out->seq_done, 1ull);
}

// worst case of one checkpoint of the region: every page dirty, one record per page
__device__ __forceinline__ u64 cc_pass_worst_bytes(const cc_region_dev& r) {
    return r.n_pages * ((u64)r.page_bytes + CC_RECORD_HEADER_BYTES) - ((u64)r.page_bytes - page_len_dev(r, r.n_pages - 1)) +
           CC_COMMIT_RECORD_BYTES;
}
