// cc_apply_parse.cuh -- a6, parallel parse of the log.
//
// The sequential definition walks record by record; every epoch ends in a 32-byte commit record.  Here the epochs
// are parsed CONCURRENTLY, with exactly the sequential result:
//   candidates  every 16-byte-aligned position of the log is tested for a commit record's signature
//               {0xFFFFFFFF, 0xFFFFFFFF, 16, crc32c(next 16 bytes)}; the positions that pass are appended to a list,
//               which a ranking step then puts in ascending order.
//               Every real commit record is on the list; a payload that happens to contain the image of a commit
//               record puts a FALSE candidate on it.
//   walk        span j = [end of candidate j-1, candidate j) is walked by one block from its start, as the sequential
//               parser would (speculative strided header reads inside a run of equal-sized records).  A span whose walk
//               lands exactly on its candidate is one committed epoch.  Spans are chained in order by a decoupled
//               look-back that carries (records, segments) of all earlier spans -- the record numbers are therefore
//               the sequential ones.  The first span of the chain that does NOT end on its candidate is where the
//               sequential parser stops (torn or structurally invalid: its partial records are kept, pending, exactly
//               as the definition holds them) -- unless the walk ran PAST its candidate (a false candidate inside a
//               payload): then, and when the candidate list overflows, `need_serial` is raised and the one-block serial
//               parser of cc_apply.cuh redoes the parse.  Correctness never depends on the speculation.
#pragma once
#include "cc_common.cuh"
#include "cc_crc.cuh"
#include "cc_ckpt.cuh"

#define CC_CAND_THREADS 256
#define CC_CAND_WARP_CAP 256u            // candidates one warp can hold for its part of a range
#define CC_WALK_THREADS 128

// span look-back word: bits 0-30 records, bits 31-61 segments, bits 62-63 flag
#define CC_SP_AGG 1ull
#define CC_SP_INC 2ull
#define CC_SP_STOP 3ull
__device__ __forceinline__ u64 sp_pack(u64 flag, u32 recs, u32 segs) { return (flag << 62) | ((u64)segs << 31) | recs; }
__device__ __forceinline__ u32 sp_recs(u64 w) { return (u32)(w & 0x7FFFFFFFull); }
__device__ __forceinline__ u32 sp_segs(u64 w) { return (u32)((w >> 31) & 0x7FFFFFFFull); }
__device__ __forceinline__ u32 sp_flag(u64 w) { return (u32)(w >> 62); }

// ---------------------------------------------------------------------------- candidates --
// grid-wide, no block barrier, no ordering: a warp tests 4 KiB of the log per step (8 independent 16-byte loads per
// lane, the scanner's loop) and appends the rare hits to an UNORDERED list with one atomic each; cc_parse_sort_phase
// then ranks the list.  (The first version kept the list ordered as it went -- ticketed ranges per block, per-warp
// ordered sub-lists, look-back over the tickets: three block barriers per 128 KiB and 78 registers held it at 2.7 TB/s,
// profiles/r02_apply_ncu.md.)  scratch: T.cand_raw[0 .. max_records].
__device__ __forceinline__ void cc_parse_cand_phase(cc_dev* dev, cc_parse_ctl* C, u32* cand_raw, u64 max_records, const u8* log, u64 n,
                                                    cc_grid g) {
    const u32 lane = threadIdx.x & 31u;
    const u64 units = n >> 4;                                    // 16-byte units of the log
    if (g.block == 0 && threadIdx.x == 0) {
        cc_apply_reset_state(dev);                               // (read by the walk phase, two launches later)
        // candidates are kept as u32 counts of 16-byte units: a log of 64 GiB or more does not fit them, and wrapped
        // offsets could coincide (the ranking below needs distinct values).  Such a log goes to the serial parser.
        if (units > 0xFFFFFFFFull) C->cand_overflow = 1;
    }
    const uint4* L = reinterpret_cast<const uint4*>(log);
    for (u64 ub = (u64)g.warp() * 256u; ub < units; ub += (u64)g.nwarps() * 256u) {
        uint4 v[8];
#pragma unroll
        for (int q = 0; q < 8; q++) {
            const u64 u = ub + 32u * q + lane;
            v[q] = (u < units) ? ld_v4(L + u) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int q = 0; q < 8; q++) {
            const u64 u = ub + 32u * q + lane;
            if ((v[q].x == CC_COMMIT_ID) && (v[q].y == CC_COMMIT_ID) && (v[q].z == 16u) && (u + 2 <= units)) {
                // rare: check the commit payload's CRC
                const uint4 pl = ld_v4(L + u + 1);
                u32 c = 0xFFFFFFFFu;
                const u32 pay[4] = {pl.x, pl.y, pl.z, pl.w};
#pragma unroll
                for (int w = 0; w < 4; w++) {
                    c ^= pay[w];
                    for (int b = 0; b < 32; b++) c = gf_mulx(c);
                }
                if ((c ^ 0xFFFFFFFFu) == v[q].w) {
                    const u32 pos = atomicAdd(&C->n_raw, 1u);
                    if ((u64)pos <= max_records) cand_raw[pos] = (u32)u;
                    else C->cand_overflow = 1;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------- sort --
// Ascending order of the candidate list by ranking: position = number of smaller candidates (they are distinct log
// offsets).  n^2 / threads comparisons out of shared-memory tiles: a hundred candidates are a few microseconds of one
// block, a hundred thousand ~0.1 ms of the whole grid -- either way far below the serial walk the ordered list saves.
// Also arms the look-back words of the walk.  scratch: T.cand[0 .. max_records], T.span_status[0 .. max_records + 1].
// The ranking is quadratic in the number of candidates (= commit records): beyond CC_SORT_MAX_CAND of them -- 2^17,
// ~0.3 ms of the whole grid -- the list is declared overflowed and the linear serial parser takes the log instead, so
// that recovery time grows with the log's bytes, not with the square of its epoch count.
#define CC_SORT_THREADS 256
#define CC_SORT_MAX_CAND (1u << 17)
__device__ __forceinline__ void cc_parse_sort_phase(cc_parse_ctl* C, const u32* cand_raw, u32* cand, u64* span_status, u64 max_records,
                                                    cc_grid g) {
    __shared__ u32 s_tile[CC_SORT_THREADS];
    const u32 tid = threadIdx.x;
    u64 n64 = C->n_raw;
    if (n64 > CC_SORT_MAX_CAND || C->cand_overflow) {             // (every block takes the same decision from n_raw)
        if (g.block == 0 && tid == 0) { C->cand_overflow = 1; C->n_cand = 0; }
        return;
    }
    if (n64 > max_records + 1) n64 = max_records + 1;
    const u32 n = (u32)n64;
    if (g.block == 0 && tid == 0) { C->n_cand = n; span_status[0] = 0; }
    for (u32 base = g.block * CC_SORT_THREADS; base < n; base += g.nblocks * CC_SORT_THREADS) {
        const u32 i = base + tid;
        const u32 mine = i < n ? cand_raw[i] : 0xFFFFFFFFu;
        u32 rank = 0;
        for (u32 t0 = 0; t0 < n; t0 += CC_SORT_THREADS) {
            __syncthreads();
            s_tile[tid] = (t0 + tid < n) ? cand_raw[t0 + tid] : 0xFFFFFFFFu;
            __syncthreads();
            const u32 m = n - t0 < CC_SORT_THREADS ? n - t0 : CC_SORT_THREADS;
            for (u32 q = 0; q < m; q++) rank += (s_tile[q] < mine) ? 1u : 0u;
        }
        if (i < n) { cand[rank] = mine; span_status[rank + 1] = 0; }
    }
}

// ---------------------------------------------------------------------------------- walk --
struct cc_walk_smem {
    u64 r_bytes[CC_MAX_REGIONS], r_pages[CC_MAX_REGIONS];
    u32 r_id[CC_MAX_REGIONS], r_P[CC_MAX_REGIONS], r_spp[CC_MAX_REGIONS];
    u64 off;                 // next unread record
    u32 nrec, nseg;          // records / segments of this span so far
    u32 pend_rid, mixed, slot, have_slot;
    u32 first_fail, first_short, width;
    u32 outcome;             // CC_WO_*
    u32 ticket;
    u32 base_recs, base_segs, dead;
    uint4 cpl;               // payload of the commit record the walk landed on
};
#define CC_WO_RUN 0u         // still walking
#define CC_WO_COMMIT 1u      // landed exactly on the span's candidate: a committed epoch
#define CC_WO_TORN 2u        // ran out of bytes: the sequential parser stops here, status OK
#define CC_WO_CORRUPT 3u     // a structural check failed: the sequential parser stops here, CC_ERR_CORRUPT
#define CC_WO_IRREGULAR 4u   // ran past the candidate (a false one): the serial parser takes over

__device__ __forceinline__ int cc_walk_find_slot(const cc_walk_smem* S, u32 rid) {
    for (int q = 0; q < CC_MAX_REGIONS; q++)
        if (S->r_id[q] == rid) return rid ? q : -1;
    return -1;
}
__device__ __forceinline__ bool cc_walk_len_ok(const cc_walk_smem* S, u32 slot, u64 page_idx, u64 len) {
    if (page_idx >= S->r_pages[slot] || len == 0) return false;
    const u64 start = page_idx * (u64)S->r_P[slot];
    if (len > S->r_bytes[slot] - start) return false;
    return (len % S->r_P[slot] == 0) || (start + len == S->r_bytes[slot]);
}

// One pass over span [start, target): WRITE = false only counts, WRITE = true also fills the record tables at
// (base_recs, base_segs).  Block-wide; the result is in S (outcome, nrec, nseg, off, pend_rid, mixed, cpl).
template <bool WRITE>
__device__ __forceinline__ void cc_walk_span(const cc_apply_tabs& T, const u8* log, u64 n, cc_walk_smem* S, u64 start, u64 target,
                                             bool has_target, u32 epoch_idx, u32 base_recs, u32 base_segs) {
    const u32 tid = threadIdx.x, nthr = blockDim.x;
    if (tid == 0) {
        S->off = start; S->nrec = 0; S->nseg = 0; S->pend_rid = 0; S->mixed = 0; S->have_slot = 0; S->outcome = CC_WO_RUN;
        S->width = has_target ? nthr : 32;      // a span with a target is bounded by it: speculate over the whole block at once
    }
    __syncthreads();
    for (;;) {
        // ---- one thread examines the record at S->off ----
        if (tid == 0) {
            const u64 off = S->off;
            u32 oc = CC_WO_RUN;
            if (has_target && off > target) oc = CC_WO_IRREGULAR;
            else if (n - off < CC_RECORD_HEADER_BYTES) oc = CC_WO_TORN;
            else {
                const uint4 h = ld_v4(reinterpret_cast<const uint4*>(log + off));
                if ((u64)h.z > n - off - CC_RECORD_HEADER_BYTES) oc = CC_WO_TORN;
                else if (h.x == CC_COMMIT_ID) {
                    // a commit header.  Its signature and CRC hold iff the position is a candidate; the only
                    // candidate the walk can meet first is its own target
                    if (has_target && off == target) {
                        const uint4 pl = ld_v4(reinterpret_cast<const uint4*>(log + off + 16));
                        const bool ok = (pl.w == S->nrec) && !S->mixed && (S->nrec == 0 || S->pend_rid == pl.z);
                        S->cpl = pl;
                        oc = ok ? CC_WO_COMMIT : CC_WO_CORRUPT;
                    } else oc = CC_WO_CORRUPT;
                } else {
                    const int slot = cc_walk_find_slot(S, h.x);
                    if (slot < 0 || !cc_walk_len_ok(S, (u32)slot, h.y, h.z)) oc = CC_WO_CORRUPT;
                    else {
                        if (S->nrec != 0 && S->pend_rid != h.x) S->mixed = 1;
                        S->pend_rid = h.x;
                        S->slot = (u32)slot;
                        S->have_slot = 1;
                        S->first_fail = nthr;
                        S->first_short = nthr + 1;
                    }
                }
            }
            S->outcome = oc;
        }
        __syncthreads();
        if (S->outcome != CC_WO_RUN) break;
        // ---- speculative run: thread t reads the header at off + t * (16 + P) ----
        const u32 slot = S->slot, rid = S->r_id[slot], spp = S->r_spp[slot];
        const u64 P = S->r_P[slot];
        const u64 stride = P + CC_RECORD_HEADER_BYTES;
        const u64 off_t = S->off + (u64)tid * stride;
        const u32 width = S->width;
        const bool active = tid < width;
        // positions at or beyond the target are never part of the run (the target itself is the commit record)
        const bool in_h = active && off_t + 16 <= n && (!has_target || off_t < target);
        uint4 h = make_uint4(0, 0, 0, 0);
        if (in_h) h = ld_v4(reinterpret_cast<const uint4*>(log + off_t));
        bool ok = in_h;
        if (ok) ok = ((u64)h.z <= n - off_t - CC_RECORD_HEADER_BYTES) && (h.x == rid) && cc_walk_len_ok(S, slot, h.y, h.z);
        const bool full = ok && ((u64)h.z == P);
        if (active && !ok) atomicMin(&S->first_fail, tid);
        else if (active && !full) { atomicMin(&S->first_fail, tid + 1); atomicMin(&S->first_short, tid + 1); }
        __syncthreads();
        const u32 run = S->first_fail < width ? S->first_fail : width;      // >= 1: record 0 was examined above
        if (WRITE && tid < run) {
            const u64 ri = (u64)base_recs + S->nrec + tid;
            if (ri < T.max_records) {
                cc_rec rec;
                rec.off = off_t; rec.page_idx = h.y; rec.len = h.z; rec.crc = h.w;
                rec.slot = slot; rec.epoch_idx = epoch_idx; rec.pad = 0;
                T.recs[ri] = rec;
                T.rec_state[ri] = 0;
                T.seg_begin[ri] = base_segs + S->nseg + tid * spp;         // only the run's last record can be short
            }
        }
        __syncthreads();
        if (tid == run - 1) {
            S->off = off_t + CC_RECORD_HEADER_BYTES + h.z;
            S->nrec += run;
            S->nseg += (run - 1) * spp + (h.z + CC_SEG_BYTES - 1) / CC_SEG_BYTES;
            if (run == width) S->width = 2 * width > nthr ? nthr : 2 * width;
        }
        __syncthreads();
    }
}

// grid-wide, blocks of CC_WALK_THREADS.  Needs: C->n_cand, T.cand, T.span_status (zeroed for 0..n_cand), A reset.
__device__ __forceinline__ void cc_parse_walk_phase(cc_dev* dev, cc_parse_ctl* C, const cc_apply_tabs& T, const u8* log, u64 n, bool first_block) {
    __shared__ cc_walk_smem S;
    cc_apply_state* A = &dev->apply;
    const u32 tid = threadIdx.x;
    if (first_block && tid == 0) C->n_raw = 0;                    // (the candidate list is sorted and counted) for the next parse
    if (C->cand_overflow) {                                       // the list is incomplete: the serial parser does it all
        if (first_block && tid == 0) C->need_serial = 1;
        return;
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
    const u32 m = C->n_cand;
    const u32 n_spans = m + 1;                                    // the last span has no candidate: the tail of the log
    for (;;) {
        __syncthreads();
        if (tid == 0) S.ticket = atomicAdd(&C->wticket, 1u);
        __syncthreads();
        const u32 j = S.ticket;
        if (j >= n_spans) break;
        const u64 start = j ? ((u64)T.cand[j - 1] << 4) + CC_COMMIT_RECORD_BYTES : 0ull;
        const bool has_target = j < m;
        const u64 target = has_target ? ((u64)T.cand[j] << 4) : 0ull;
        cc_walk_span<false>(T, log, n, &S, start, target, has_target, j, 0, 0);
        const u32 oc = S.outcome, nrec = S.nrec, nseg = S.nseg;
        // ---- chain: records / segments of all earlier spans; dead if an earlier span stopped the parse.  Warp-wide
        //      look-back: 32 predecessors per step (one thread walking back word by word made span 99 wait through up to
        //      99 dependent loads) ----
        if (tid < 32) {
            const u32 lane = tid;
            if (j != 0 && lane == 0)
                st_release_gpu_u64(&T.span_status[j], sp_pack(oc == CC_WO_COMMIT ? CC_SP_AGG : CC_SP_STOP, nrec, nseg));
            u32 br = 0, bs = 0, dead = 0;
            int base = (int)j - 1;
            while (base >= 0) {
                const int q = base - (int)lane;
                u64 s = sp_pack(CC_SP_INC, 0, 0);                 // virtual span -1: inclusive (0, 0)
                if (q >= 0) s = ld_acquire_gpu_u64(&T.span_status[q]);
                const u32 f = sp_flag(s);
                const u32 nr = __ballot_sync(0xFFFFFFFFu, f == 0);
                const u32 term = __ballot_sync(0xFFFFFFFFu, f == CC_SP_INC || f == CC_SP_STOP);
                const u32 first_nr = nr ? (u32)__ffs(nr) - 1u : 32u;
                const u32 first_t = term ? (u32)__ffs(term) - 1u : 32u;
                if (first_nr < first_t) { __nanosleep(20); continue; }     // a nearer predecessor has not published yet
                const u32 upto = first_t < 32u ? first_t : 31u;
                const bool in = lane <= upto;
                const u32 tf = __shfl_sync(0xFFFFFFFFu, f, upto);
                if (first_t < 32u && tf == CC_SP_STOP) { dead = 1; break; }
                br += __reduce_add_sync(0xFFFFFFFFu, in ? sp_recs(s) : 0u);
                bs += __reduce_add_sync(0xFFFFFFFFu, in ? sp_segs(s) : 0u);
                if (first_t < 32u) break;                         // reached an inclusive word
                base -= 32;
            }
            if (lane == 0) { S.base_recs = br; S.base_segs = bs; S.dead = dead; }
        }
        __syncthreads();
        if (S.dead) {                                             // something before this span ended the parse
            if (tid == 0) st_release_gpu_u64(&T.span_status[j], sp_pack(CC_SP_STOP, 0, 0));
            continue;
        }
        const u32 br = S.base_recs, bs = S.base_segs;
        const bool overflow = (u64)br + nrec > T.max_records || (oc == CC_WO_COMMIT && (u64)j >= T.max_records);
        if (!overflow && oc != CC_WO_IRREGULAR && nrec != 0)
            cc_walk_span<true>(T, log, n, &S, start, target, has_target, j, br, bs);
        if (tid == 0) {
            if (oc == CC_WO_COMMIT && !overflow) {
                cc_epoch_ent e;
                e.off_after = target + CC_COMMIT_RECORD_BYTES;
                e.epoch_no = (u64)S.cpl.x | ((u64)S.cpl.y << 32);
                e.rec_end = br + nrec;
                e.slot = S.have_slot ? S.slot : 0xFFFFFFFFu;
                e.pending = nrec;
                e.pad = 0;
                T.epochs[j] = e;
                if (nrec != 0) atomicMax(&dev->compactor.region_last[S.slot], j + 1);
                __threadfence();
                st_release_gpu_u64(&T.span_status[j], sp_pack(CC_SP_INC, br + nrec, bs + nseg));
            } else {
                // this span ends the parse: totals, and why
                if (oc == CC_WO_IRREGULAR) C->need_serial = 1;
                if (overflow) A->scratch_overflow = 1;
                if (oc == CC_WO_CORRUPT) A->struct_fail = 1;
                const u32 kept = (overflow || oc == CC_WO_IRREGULAR) ? 0u : nrec;
                A->n_recs = br + kept;
                A->n_epochs = j;
                T.seg_begin[br + kept] = bs + (kept ? nseg : 0u);      // table has max_records + 1 entries
                __threadfence();
                st_release_gpu_u64(&T.span_status[j], sp_pack(CC_SP_STOP, 0, 0));
            }
        }
    }
}
