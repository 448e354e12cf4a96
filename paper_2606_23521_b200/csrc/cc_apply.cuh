// cc_apply.cuh -- a6, the recovery applier ("fn.apply(aof_read(epoch))", L221
// "Recovery ignores any suffix without a commit marker", L227 "replays ... committed AOF suffix").
//
// The sequential definition (walk record by record; hold page records pending until their commit
// validates; apply epochs in log order) is reproduced exactly by data-parallel phases:
//   parse    cc_apply_parse.cuh: candidate commit records by signature search over the whole log, then every
//            epoch walked by its own block, chained by look-back (sequential record numbers); a one-block serial
//            walk (below) is the fallback when the speculation does not hold (false candidates, list overflow).
//            Inside an epoch all full-page records of a region have the same stride 16+P, so a walk reads
//            blockDim headers speculatively per step and accepts the leading run that is structurally valid.
//            The walk stops at the first torn or structurally invalid record, exactly where the definition stops.
//   validate every 4 KiB payload segment is CRC'd by a warp; a record whose CRC differs lowers
//            first_bad_rec (atomicMin).  The last block then resolves the committed prefix:
//            the epochs whose records all precede the first failed check.
//   latest   atomicMax(latest[page], rec+1) over the committed records (last record wins).
//   scatter  a segment is copied into the live page and the shadow only if its record is the
//            page's latest.
//   cleanup  latest[] back to zero; result written.
#pragma once
#include "cc_common.cuh"
#include "cc_crc.cuh"

struct cc_apply_tabs {      // carved out of the attached scratch
    cc_rec* recs;
    cc_epoch_ent* epochs;   // max_records + 1
    u64* rec_state;         // per-record {done-mask or count | CRC accumulator} (crc_record_combine)
    u32* seg_begin;         // per-record first segment number (+ one trailing total)
    u32* cand;              // max_records + 1: candidate commit records, log offset / 16, ascending
    u32* cand_raw;          // max_records + 1: the same as found (unordered)
    u64* span_status;       // max_records + 2: look-back words of the epoch walk
    u64 max_records;
};

__device__ __forceinline__ int cc_find_slot(const cc_dev* dev, u32 rid) {
    for (int s = 0; s < CC_MAX_REGIONS; s++)
        if (dev->region_used[s] && dev->regions[s].region_id == rid) return s;
    return -1;
}

// A page record may carry a run of consecutive pages (PAPER.md:L221 run-length encoding; reading #38):
// (page_idx, len) is well-formed iff it denotes a whole number (>= 1) of pages inside the region.
__device__ __forceinline__ bool cc_rec_len_ok(const cc_region_dev& r, u64 page_idx, u64 len) {
    if (page_idx >= r.n_pages || len == 0) return false;
    const u64 start = page_idx * (u64)r.page_bytes;
    if (len > r.bytes - start) return false;
    return (len % r.page_bytes == 0) || (start + len == r.bytes);
}
__device__ __forceinline__ u32 cc_rec_pages(const cc_region_dev& r, u32 len) {
    return (u32)(((u64)len + r.page_bytes - 1) / r.page_bytes);
}
// 0xFFFFFFFF * x^(8*len): the CRC init term of a record of len bytes
__device__ __forceinline__ u32 cc_crc_init_term(const cc_dev* dev, const cc_region_dev& r, u32 len) {
    if (len == r.page_bytes) return r.crc_init_full;
    if ((u64)len == page_len_dev(r, r.n_pages - 1)) return r.crc_init_tail;
    return gf_mul(0xFFFFFFFFu, gf_xpow_bytes(dev->crc.xp, len));
}

#define CC_PA_STOP 0u
#define CC_PA_NEXT 1u
#define CC_PA_RUN 2u

struct cc_parse_smem {
    // the region table, copied once: the walk is a chain of dependent decisions, and every global load in it is
    // a round trip to L2 (a few hundred ns) -- with the table in shared memory an epoch costs one load round
    u64 r_bytes[CC_MAX_REGIONS], r_pages[CC_MAX_REGIONS];
    u32 r_id[CC_MAX_REGIONS], r_P[CC_MAX_REGIONS], r_spp[CC_MAX_REGIONS];       // r_id = 0: slot unused
    u64 off;                // offset of the next unread record
    u32 action, slot, first_fail, first_short, nrecs, nepochs, pending, pend_rid, mixed, segs;
    u32 width;              // speculation width of the next step: about the size of the previous epoch (reads far beyond
                            // the epoch's end are wasted and only lengthen the step's slowest load)
    u32 pre;                // the record at `off` has already been examined (action / slot are set)
    u32 cand;               // thread whose speculative header sits right after the accepted run (or 0xFFFFFFFF)
};

__device__ __forceinline__ int cc_parse_find_slot(const cc_parse_smem* S, u32 rid) {
    for (int q = 0; q < CC_MAX_REGIONS; q++)
        if (S->r_id[q] == rid) return rid ? q : -1;
    return -1;
}
__device__ __forceinline__ bool cc_parse_len_ok(const cc_parse_smem* S, u32 slot, u64 page_idx, u64 len) {
    if (page_idx >= S->r_pages[slot] || len == 0) return false;
    const u64 start = page_idx * (u64)S->r_P[slot];
    if (len > S->r_bytes[slot] - start) return false;
    return (len % S->r_P[slot] == 0) || (start + len == S->r_bytes[slot]);
}

// Examine the record at S->off (one thread).  A commit record is validated and its epoch pushed (CC_PA_NEXT); a
// page record opens a speculative run (CC_PA_RUN); anything torn or invalid stops the walk (CC_PA_STOP), exactly
// where the sequential definition stops.  pre_h / pre_pl: the header / the 16 bytes after it, if already loaded.
__device__ __forceinline__ u32 cc_parse_examine(cc_dev* dev, const cc_apply_tabs& T, const u8* log, u64 n, cc_parse_smem* S, u32 nthr,
                                                bool have_h, uint4 pre_h, bool have_pl, uint4 pre_pl) {
    cc_apply_state* A = &dev->apply;
    const u64 off = S->off;
    if (n - off < CC_RECORD_HEADER_BYTES) return CC_PA_STOP;                               // torn
    const uint4 h = have_h ? pre_h : ld_v4(reinterpret_cast<const uint4*>(log + off));
    if ((u64)h.z > n - off - CC_RECORD_HEADER_BYTES) return CC_PA_STOP;                    // torn
    if (h.x == CC_COMMIT_ID) {
        bool ok = (h.y == CC_COMMIT_ID) && (h.z == 16u);
        uint4 pl = make_uint4(0, 0, 0, 0);
        if (ok) {
            pl = have_pl ? pre_pl : ld_v4(reinterpret_cast<const uint4*>(log + off + 16));
            u32 pay[4] = {pl.x, pl.y, pl.z, pl.w};
            ok = crc_serial(&dev->crc, reinterpret_cast<const u8*>(pay), 16) == h.w;
            ok = ok && (pl.w == S->pending) && !S->mixed && (S->pending == 0 || S->pend_rid == pl.z);
        }
        if (!ok) { A->struct_fail = 1; return CC_PA_STOP; }
        if (S->nepochs >= T.max_records) { A->scratch_overflow = 1; return CC_PA_STOP; }
        {
            const int cs = S->pending != 0 ? cc_parse_find_slot(S, pl.z) : -1;
            if (cs >= 0) dev->compactor.region_last[cs] = S->nepochs + 1;       // for the log compactor: last epoch per region
            cc_epoch_ent e;
            e.off_after = off + CC_COMMIT_RECORD_BYTES;
            e.epoch_no = (u64)pl.x | ((u64)pl.y << 32);
            e.rec_end = S->nrecs;
            e.slot = cs >= 0 ? (u32)cs : 0xFFFFFFFFu;
            e.pending = S->pending;
            e.pad = 0;
            T.epochs[S->nepochs] = e;
        }
        S->nepochs++;
        S->width = S->pending + 16u < 32u ? 32u : (S->pending + 16u > nthr ? nthr : S->pending + 16u);
        S->pending = 0; S->mixed = 0;
        S->off = off + CC_COMMIT_RECORD_BYTES;
        return CC_PA_NEXT;
    }
    const int slot = cc_parse_find_slot(S, h.x);
    if (slot < 0) { A->struct_fail = 1; return CC_PA_STOP; }
    if (!cc_parse_len_ok(S, (u32)slot, h.y, h.z)) { A->struct_fail = 1; return CC_PA_STOP; }
    if (S->pending != 0 && S->pend_rid != h.x) S->mixed = 1;
    S->pend_rid = h.x;
    S->slot = (u32)slot;
    S->first_fail = nthr;
    S->first_short = nthr + 1;
    return CC_PA_RUN;
}

// One block walks the log.  Steady state is ONE step per epoch: every thread speculatively reads the header at its
// stride position (and, if that is a commit record, the 32 bytes after it); the leading run of full single-page records is accepted; the thread
// sitting right behind the run usually holds the epoch's commit record -- it validates it from the bytes it
// already has and examines the first header of the next epoch (also already loaded), so that the next step can
// start its speculative reads at once.
// One thread, before any parse phase: the applier's state for a new log.
__device__ __forceinline__ void cc_apply_reset_state(cc_dev* dev) {
    cc_apply_state* A = &dev->apply;
    A->n_recs = 0; A->n_epochs = 0;
    A->struct_fail = 0; A->scratch_overflow = 0; A->first_bad_rec = 0xFFFFFFFFu; A->validate_done = 0;
    A->n_commit_recs = 0; A->n_commit_epochs = 0; A->consumed = 0; A->status = CC_OK; A->final_done = 0;
    A->t_start_ns = globaltimer_ns();
    for (int s = 0; s < CC_MAX_REGIONS; s++) dev->compactor.region_last[s] = 0;
}

// The serial walk: ONE block.  It is the fallback of the parallel parse (cc_apply_parse.cuh) and runs only when
// that raised need_serial (force = false), or as the parser proper (force = true).
__device__ __forceinline__ void cc_apply_parse_phase(cc_dev* dev, const cc_apply_tabs& T, const u8* log, u64 n, bool force) {
    __shared__ cc_parse_smem S;
    cc_apply_state* A = &dev->apply;
    const u32 tid = threadIdx.x, nthr = blockDim.x;
    if (!force && !dev->parse.need_serial) return;
    __syncthreads();                             // (every thread has read need_serial before it is touched)
    if (tid == 0) {
        S.off = 0; S.nrecs = 0; S.nepochs = 0; S.pending = 0; S.pend_rid = 0; S.mixed = 0; S.segs = 0; S.pre = 0;
        S.action = CC_PA_STOP; S.cand = 0xFFFFFFFFu; S.width = nthr < 128u ? nthr : 128u;
        const u64 t0 = A->t_start_ns;
        cc_apply_reset_state(dev);
        if (!force) A->t_start_ns = t0;
    }
    if (tid < CC_MAX_REGIONS) {
        const bool used = dev->region_used[tid] != 0;
        const cc_region_dev& rg = dev->regions[tid];
        S.r_id[tid] = used ? rg.region_id : 0u;
        S.r_P[tid] = used ? rg.page_bytes : 1u;
        S.r_spp[tid] = used ? rg.spp : 1u;
        S.r_bytes[tid] = used ? rg.bytes : 0ull;
        S.r_pages[tid] = used ? rg.n_pages : 0ull;
    }
    __syncthreads();
    for (;;) {
        if (tid == 0) {
            if (!S.pre) S.action = cc_parse_examine(dev, T, log, n, &S, nthr, false, make_uint4(0, 0, 0, 0), false, make_uint4(0, 0, 0, 0));
            S.pre = 0;
        }
        __syncthreads();
        const u32 action = S.action;
        if (action == CC_PA_STOP) break;
        if (action == CC_PA_RUN) {
            const u32 slot = S.slot, rid = S.r_id[slot], spp = S.r_spp[slot];
            const u64 P = S.r_P[slot];
            const u64 stride = P + CC_RECORD_HEADER_BYTES;
            const u64 off_t = S.off + (u64)tid * stride;
            const u32 width = S.width;
            uint4 h = make_uint4(0, 0, 0, 0), pl = h, nx = h;
            const bool active = tid < width;
            const bool in_h = active && off_t + 16 <= n, in_pl = active && off_t + 32 <= n, in_nx = active && off_t + 48 <= n;
            bool ok = in_h;
            if (in_h) h = ld_v4(reinterpret_cast<const uint4*>(log + off_t));
            const bool commit_here = in_pl && h.x == CC_COMMIT_ID;      // (normally one thread per step)
            if (commit_here) pl = ld_v4(reinterpret_cast<const uint4*>(log + off_t + 16));           // the commit record's payload
            if (commit_here && in_nx) nx = ld_v4(reinterpret_cast<const uint4*>(log + off_t + 32));  // ... and the header after it
            if (ok) ok = ((u64)h.z <= n - off_t - CC_RECORD_HEADER_BYTES) && (h.x == rid) && cc_parse_len_ok(&S, slot, h.y, h.z);
            // a short (tail) page or a multi-page run record is valid but breaks the stride: it may only END a run
            const bool full = ok && ((u64)h.z == P);
            if (active && !ok) atomicMin(&S.first_fail, tid);
            else if (active && !full) { atomicMin(&S.first_fail, tid + 1); atomicMin(&S.first_short, tid + 1); }
            __syncthreads();
            const u32 run = S.first_fail < width ? S.first_fail : width;    // >= 1: record 0 was examined before
            const u32 base = S.nrecs;
            const bool overflow = (u64)base + run > T.max_records;
            if (!overflow && tid < run) {
                cc_rec rec;
                rec.off = off_t; rec.page_idx = h.y; rec.len = h.z; rec.crc = h.w;
                rec.slot = slot; rec.epoch_idx = S.nepochs; rec.pad = 0;
                T.recs[base + tid] = rec;
                T.rec_state[base + tid] = 0;
                T.seg_begin[base + tid] = S.segs + tid * spp;          // only the run's last record can be short
            }
            const u32 first_short = S.first_short;
            __syncthreads();
            if (!overflow && tid == run - 1) {                         // the run's last record knows where the run ends
                S.off = off_t + CC_RECORD_HEADER_BYTES + h.z;
                S.nrecs = base + run;
                S.pending += run;
                S.segs += (run - 1) * spp + (h.z + CC_SEG_BYTES - 1) / CC_SEG_BYTES;
                // the thread right behind the run sits on the next record iff the run ended on a full page
                S.cand = (run < width && first_short > run) ? run : 0xFFFFFFFFu;
                if (run == width) S.width = 2 * width > nthr ? nthr : 2 * width;      // the epoch is longer than expected
            }
            if (overflow && tid == 0) { A->scratch_overflow = 1; S.action = CC_PA_STOP; S.cand = 0xFFFFFFFFu; }
            __syncthreads();
            if (S.action == CC_PA_STOP) break;
            if (tid == S.cand && in_h && h.x == CC_COMMIT_ID) {
                // S.off == off_t here.  Commit from the preloaded bytes, then the next epoch's first header.
                u32 act = cc_parse_examine(dev, T, log, n, &S, nthr, true, h, commit_here, pl);
                if (act == CC_PA_NEXT) act = cc_parse_examine(dev, T, log, n, &S, nthr, commit_here && in_nx, nx, false, make_uint4(0, 0, 0, 0));
                if (act != CC_PA_NEXT) { S.action = act; S.pre = 1; }      // NEXT again (an empty epoch): thread 0 goes on
            }
            __syncthreads();
        }
    }
    if (tid == 0) {
        A->n_recs = S.nrecs;
        A->n_epochs = S.nepochs;
        T.seg_begin[S.nrecs] = S.segs;          // table has max_records + 1 entries
        __threadfence();
    }
}

#include "cc_apply_parse.cuh"

// warp-cooperative search: largest rec with seg_begin[rec] <= item, rec in [0, n)
__device__ __forceinline__ u32 cc_find_rec(const u32* seg_begin, u32 n, u32 item, u32 lane) {
    u32 lo = 0, hi = n;
    while (hi - lo > 1) {
        const u32 step = (hi - lo + 31) / 32;
        const u32 idx = lo + lane * step;
        const bool le = (idx < hi) && (seg_begin[idx] <= item);
        const u32 cnt = __popc(__ballot_sync(0xFFFFFFFFu, le));     // >= 1 (lane 0)
        lo = lo + (cnt - 1) * step;
        hi = min(lo + step, hi);
    }
    return lo;
}

// CRC32C contribution of segment c of record ri (in every lane).
template <class SM>
__device__ __forceinline__ u32 cc_apply_segment_crc(cc_dev* dev, SM* cs, const u8* log, const cc_rec& rec, u32 c, u32 lane) {
    constexpr int U = 8;
    const u64 so = (u64)c * CC_SEG_BYTES;
    const u64 rem = rec.len - so;
    const u32 seg_len = (u32)(rem < CC_SEG_BYTES ? rem : CC_SEG_BYTES);
    const u32 nv = seg_len >> 4;
    const uint4* src = reinterpret_cast<const uint4*>(log + rec.off + CC_RECORD_HEADER_BYTES + so);
    uint4 v[U];
#pragma unroll
    for (int u = 0; u < U; u++) {
        const u32 j = lane + 32 * u;
        v[u] = (j < nv) ? ld_v4(src + j) : make_uint4(0, 0, 0, 0);
    }
    return crc_segment_warp<U>(cs, &dev->crc, v, nv, rem - seg_len, lane);
}
// Segments c0 .. c0 + cn - 1 of record ri are checked (contrib = XOR of their contributions): the warp that completes the
// record compares with the header's CRC.
__device__ __forceinline__ void cc_apply_record_verdict(cc_dev* dev, const cc_apply_tabs& T, u32 ri, const cc_rec& rec, u32 c0, u32 cn,
                                                        u32 contrib, u32 lane) {
    if (lane != 0) return;
    const u32 nseg = (rec.len + CC_SEG_BYTES - 1) / CC_SEG_BYTES;
    u32 acc = 0;
    if (crc_record_combine_n(&T.rec_state[ri], nseg, c0, cn, contrib, &acc)) {
        const u32 it = cc_crc_init_term(dev, dev->regions[rec.slot], rec.len);
        if (crc_finalize(acc, it) != rec.crc) atomicMin(&dev->apply.first_bad_rec, ri);
    }
}

// Segment c of record ri into the live page and the shadow -- if the record is the page's LATEST one.  A segment lies
// inside one page when pages are whole multiples of 4 KiB (or the record is a single page); otherwise the check is per
// 16-byte vector.
__device__ __forceinline__ void cc_apply_scatter_segment(cc_dev* dev, const u8* log, u32 ri, const cc_rec& rec, u32 c, u32 lane) {
    constexpr int U = 8;
    const cc_region_dev& r = dev->regions[rec.slot];
    const u64 so = (u64)c * CC_SEG_BYTES;
    const u64 rem = rec.len - so;
    const u32 nv = (u32)(rem < CC_SEG_BYTES ? rem : CC_SEG_BYTES) >> 4;
    const bool one_page = (r.page_bytes % CC_SEG_BYTES == 0) || rec.len <= r.page_bytes;
    if (one_page && r.latest[rec.page_idx + (u32)(so / r.page_bytes)] != ri + 1) return;
    const uint4* src = reinterpret_cast<const uint4*>(log + rec.off + CC_RECORD_HEADER_BYTES + so);
    const u64 dst_off = (u64)rec.page_idx * r.page_bytes + so;
    uint4* d0 = reinterpret_cast<uint4*>(r.base + dst_off);
    uint4* d1 = reinterpret_cast<uint4*>(r.shadow + dst_off);
    uint4 v[U];
    bool take[U];
#pragma unroll
    for (int u = 0; u < U; u++) {
        const u32 j = lane + 32 * u;
        take[u] = j < nv;
        if (take[u] && !one_page) take[u] = r.latest[rec.page_idx + (u32)((so + 16ull * j) / r.page_bytes)] == ri + 1;
        if (take[u]) v[u] = ld_v4(src + j);
    }
#pragma unroll
    for (int u = 0; u < U; u++) {
        const u32 j = lane + 32 * u;
        if (take[u]) { st_stream(d0 + j, v[u]); if (r.shadow) st_stream(d1 + j, v[u]); }
    }
}

#define CC_APPLY_CHUNK 4u       // consecutive 4 KiB segments one warp takes per search of the record table

// One thread, once every CRC verdict is in: the committed prefix = the epochs whose records all precede the first failed
// check; status; and the parallel parse re-armed for the next log.
__device__ __forceinline__ void cc_apply_resolve(cc_dev* dev, const cc_apply_tabs& T) {
    cc_apply_state* A = &dev->apply;
    const u32 f = A->first_bad_rec;           // 0xFFFFFFFF if every CRC matched
    const u32 ne = A->n_epochs;
    u32 lo = 0, hi = ne;                      // epochs are ordered by rec_end: count those with rec_end <= f
    while (lo < hi) {
        const u32 mid = (lo + hi) >> 1;
        if (T.epochs[mid].rec_end <= f) lo = mid + 1; else hi = mid;
    }
    int32_t st = CC_OK;
    if (f != 0xFFFFFFFFu || A->struct_fail) st = CC_ERR_CORRUPT;
    u32 E = lo;
    if (A->scratch_overflow) { st = CC_ERR_SCRATCH; E = 0; }
    A->n_commit_epochs = E;
    A->n_commit_recs = E ? T.epochs[E - 1].rec_end : 0;
    A->consumed = E ? T.epochs[E - 1].off_after : 0;
    A->status = st;
    dev->parse.cand_overflow = 0;             // re-arm the parallel parse for the next log
    dev->parse.need_serial = 0;
}

template <class SM>
__device__ __forceinline__ void cc_apply_validate_phase(cc_dev* dev, const cc_apply_tabs& T, SM* cs,
                                                        const u8* log, cc_grid g, bool init_tables) {
    cc_apply_state* A = &dev->apply;
    const u32 n_recs = A->n_recs;
    const u32 lane = threadIdx.x & 31u;
    if (g.block == 0 && threadIdx.x == 0) dev->parse.wticket = 0;      // (the walk is over) for the next parse
    if (n_recs != 0 && !A->scratch_overflow) {
        if (init_tables) cc_crc_smem_init(cs, &dev->crc);
        const u32 n_items = T.seg_begin[n_recs];
        const u32 n_chunks = (n_items + CC_APPLY_CHUNK - 1) / CC_APPLY_CHUNK;
        // from the END of the log to its head: the candidate search has just streamed the log front to back, so
        // its tail is what the L2 still holds
        for (u32 ch = g.warp(); ch < n_chunks; ch += g.nwarps()) {
            const u32 item0 = (n_chunks - 1 - ch) * CC_APPLY_CHUNK;
            const u32 item1 = item0 + CC_APPLY_CHUNK < n_items ? item0 + CC_APPLY_CHUNK : n_items;
            u32 ri = cc_find_rec(T.seg_begin, n_recs, item0, lane);
            cc_rec rec = T.recs[ri];
            u32 sb = T.seg_begin[ri], next = T.seg_begin[ri + 1];
            // consecutive segments of one record are handed in together: one 64-bit combine per record and chunk
            u32 c0 = item0 - sb, cn = 0, contrib = 0;
            for (u32 item = item0; item < item1; item++) {
                if (item >= next) {
                    cc_apply_record_verdict(dev, T, ri, rec, c0, cn, contrib, lane);
                    while (item >= next) { ri++; rec = T.recs[ri]; sb = next; next = T.seg_begin[ri + 1]; }
                    c0 = item - sb; cn = 0; contrib = 0;
                }
                contrib ^= cc_apply_segment_crc(dev, cs, log, rec, item - sb, lane);
                cn++;
            }
            cc_apply_record_verdict(dev, T, ri, rec, c0, cn, contrib, lane);
        }
    }
    // last block resolves the committed prefix
    __shared__ u32 s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(&A->validate_done, 1u) == g.nblocks - 1) ? 1u : 0u;
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        __threadfence();
        cc_apply_resolve(dev, T);
        A->validate_done = 0;
        __threadfence();
    }
}

__device__ __forceinline__ void cc_apply_latest_phase(cc_dev* dev, const cc_apply_tabs& T, cc_grid g) {
    const u32 n = dev->apply.n_commit_recs;
    for (u32 i = g.block * blockDim.x + threadIdx.x; i < n; i += g.nblocks * blockDim.x) {
        const cc_rec rec = T.recs[i];
        const cc_region_dev& r = dev->regions[rec.slot];
        const u32 m = cc_rec_pages(r, rec.len);
        for (u32 q = 0; q < m; q++) atomicMax(&r.latest[rec.page_idx + q], i + 1);
    }
}

__device__ __forceinline__ void cc_apply_scatter_phase(cc_dev* dev, const cc_apply_tabs& T, const u8* log, cc_grid g) {
    const u32 n = dev->apply.n_commit_recs;
    if (n == 0) return;
    const u32 lane = threadIdx.x & 31u;
    const u32 n_items = T.seg_begin[n];
    const u32 n_chunks = (n_items + CC_APPLY_CHUNK - 1) / CC_APPLY_CHUNK;
    for (u32 ch = g.warp(); ch < n_chunks; ch += g.nwarps()) {
        const u32 item0 = ch * CC_APPLY_CHUNK;
        const u32 item1 = item0 + CC_APPLY_CHUNK < n_items ? item0 + CC_APPLY_CHUNK : n_items;
        u32 ri = cc_find_rec(T.seg_begin, n, item0, lane);
        cc_rec rec = T.recs[ri];
        u32 sb = T.seg_begin[ri], next = T.seg_begin[ri + 1];
        for (u32 item = item0; item < item1; item++) {
            while (item >= next) { ri++; rec = T.recs[ri]; sb = next; next = T.seg_begin[ri + 1]; }
            cc_apply_scatter_segment(dev, log, ri, rec, item - sb, lane);
        }
    }
}

__device__ __forceinline__ void cc_apply_cleanup_phase(cc_dev* dev, const cc_apply_tabs& T, cc_grid g, cc_result* out,
                                                       u32 kind) {
    cc_apply_state* A = &dev->apply;
    const u32 n = A->n_commit_recs;
    for (u32 i = g.block * blockDim.x + threadIdx.x; i < n; i += g.nblocks * blockDim.x) {
        const cc_rec rec = T.recs[i];
        const cc_region_dev& r = dev->regions[rec.slot];
        const u32 m = cc_rec_pages(r, rec.len);
        for (u32 q = 0; q < m; q++) r.latest[rec.page_idx + q] = 0;
    }
    if (g.block == 0 && threadIdx.x == 0 && out) {
        out->n_dirty = n;
        out->bytes = A->consumed;
        out->log_offset_after = A->consumed;
        out->epoch = A->n_commit_epochs;
        out->status = A->status;
        out->flags = kind;
        out->t_start_ns = A->t_start_ns;
        out->t_end_ns = globaltimer_ns();
        __threadfence_system();
        st_release_sys_u64(&out->seq_done, 1ull);
    }
}
