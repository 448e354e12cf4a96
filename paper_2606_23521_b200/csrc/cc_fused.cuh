// cc_fused.cuh -- fused single pass over the region (SURVEY.md 8f #2 "scan -> offset (decoupled
// look-back) -> gather in one kernel"): a1 + a2 + (when it is safe) a3 + a5 in ONE sweep, with no
// block-level synchronisation at all -- the unit of work is a WARP TILE.
//
// Warp tiles of ~32 KiB of region (1..32 whole pages; measured: 64 KiB tiles make the warps that found dirty pages wait
// longer for their predecessors -- a 256 MiB / 4 KiB-page task in the worker took 179 us, 116 us with 16-32 KiB tiles) are handed out by ticket.  A warp scans its
// tile page by page (same 16-byte streaming loads as cc_scan_phase, with an early-out per page once
// a difference is found), keeps the tile's dirty mask in a register, publishes the tile's dirty
// count and resolves the number of dirty pages in all earlier tiles by a warp-wide decoupled
// look-back (32 predecessors per step).  That number is the record index of its first dirty page,
// so D[] comes out ascending and record i sits at W + i*(16+P) exactly as in the three-kernel path.
// The warp then gathers its own dirty pages right away: one read per segment -> log payload, shadow,
// CRC32C (running Horner over the page's segments in a register: no atomics), header -- while the
// other warps keep scanning.  The latency/ALU-bound record writer hides under the HBM-bound scan,
// and with a pinned host log the host-link transfer overlaps the scan instead of following it.
//
// All-or-nothing (reading #10) without a second pass: records are written inline only if the WORST
// case (every page dirty) fits behind the current write offset; otherwise this pass only produces
// D[], k and the plan, and the classic gather writes the records.  Either way cc_gather_phase
// follows: with inline_done set it merely appends the commit record, publishes and fills the result.
#pragma once
#include "cc_common.cuh"
#include "cc_crc.cuh"
#include "cc_ckpt.cuh"

// Warp-wide decoupled look-back: sum of the dirty counts of tiles [0, t).  The status words are read and
// written with RELAXED gpu-scope accesses: the count a word carries is the whole message (nothing else a tile
// wrote is read by another tile inside this kernel), and a release here would make the publishing warp wait
// for its earlier record stores -- over the host link with a pinned log -- and stall every tile behind it.  blocking = false gives up
// (returns false) as soon as a predecessor that has not published yet is met before an inclusive one.
__device__ __forceinline__ bool cc_fused_lookback(const u64* status, u32 run, u32 t, u32 lane, bool blocking, u32* excl_out) {
    u32 excl = 0;
    int base = (int)t - 1;
    for (;;) {
        const int j = base - (int)lane;
        u64 s = lb_pack(run, CC_LB_INC, 0);                 // virtual tile -1: inclusive sum 0
        if (j >= 0) s = ld_relaxed_gpu_u64(&status[j]);
        const u32 flag = (u32)(s >> 32) & 3u;
        const bool valid = ((u32)(s >> 34) == run) && flag != 0;
        const u32 inv = __ballot_sync(0xFFFFFFFFu, !valid);
        const u32 inc = __ballot_sync(0xFFFFFFFFu, valid && flag == (u32)CC_LB_INC);
        const u32 first_inv = inv ? (u32)__ffs(inv) - 1u : 32u;
        const u32 first_inc = inc ? (u32)__ffs(inc) - 1u : 32u;
        if (first_inc < first_inv) {                        // nearest inclusive predecessor, all nearer ones valid
            excl += __reduce_add_sync(0xFFFFFFFFu, lane <= first_inc ? (u32)s : 0u);
            *excl_out = excl;
            return true;
        }
        if (first_inv < 32u) {                              // someone has not published yet
            if (!blocking) return false;
            __nanosleep(40);
            continue;
        }
        excl += __reduce_add_sync(0xFFFFFFFFu, (u32)s);     // 32 aggregates: keep walking
        base -= 32;
    }
}

// acc * x^(8*4096): lane i contributes bit (31-i) of acc times pow_lane = x^(8*4096) * x^i.
__device__ __forceinline__ u32 cc_warp_mul_seg(u32 acc, u32 pow_lane, u32 lane) {
    u32 term = ((acc >> (31 - lane)) & 1u) ? pow_lane : 0u;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) term ^= __shfl_xor_sync(0xFFFFFFFFu, term, o);
    return term;
}

__device__ __forceinline__ void cc_fused_phase(const cc_region_dev& r, cc_dev* dev, cc_crc_smem* cs, u32 mode, u64 epoch,
                                               bool init_tables) {
    constexpr int U = 8;
    cc_ws_hdr* h = r.hdr;
    cc_log_dev* log = &dev->log;
    const u32 lane = threadIdx.x & 31u;
    const u32 P = r.page_bytes, TP = r.ftile_pages, nt = r.n_ftiles;
    const u32 run = h->frun & 0x3FFFFFFFu;
    const u64 W0 = log->W;
    const u64 rec_stride = (u64)P + CC_RECORD_HEADER_BYTES;
    // worst case: every page dirty (the last one may be short)
    const u64 worst = r.n_pages * rec_stride - ((u64)P - page_len_dev(r, r.n_pages - 1)) + CC_COMMIT_RECORD_BYTES;
    const bool inline_ok = (mode == CC_MODE_CHECKPOINT) && log->buf != nullptr && W0 + worst <= log->capacity;
    const bool has_shadow = r.shadow != nullptr;
    if (inline_ok && init_tables) cc_crc_smem_init(cs, &dev->crc);
    if (blockIdx.x == 0 && threadIdx.x == 0) h->t_start_ns = globaltimer_ns();
    const u32 pow_lane = dev->crc.seg_pow[32 + lane];

    for (;;) {
        u32 t = 0;
        if (lane == 0) t = atomicAdd(&h->fticket, 1u);
        t = __shfl_sync(0xFFFFFFFFu, t, 0);
        if (t >= nt) break;
        const u64 p0 = (u64)t * TP;
        const u32 np = (u32)((r.n_pages - p0) < TP ? (r.n_pages - p0) : TP);
        // ---- a1: scan the tile page by page; stop reading a page at its first differing segment ----
        u32 mask = 0;
        for (u32 pl = 0; pl < np; pl++) {
            const u64 p = p0 + pl;
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
            if (dirty) mask |= 1u << pl;
        }
        // ---- a2: rank of this tile's dirty pages among all dirty pages ----
        const u32 cnt = __popc(mask);
        const bool last = (t == nt - 1);
        u32 excl = 0;
        if (cnt == 0 && !last) {
            // nothing to place: publish, upgrading to an inclusive sum only if that costs no waiting
            const bool got = cc_fused_lookback(r.flb_status, run, t, lane, false, &excl);
            if (lane == 0) st_relaxed_gpu_u64(&r.flb_status[t], got ? lb_pack(run, CC_LB_INC, excl) : lb_pack(run, CC_LB_AGG, 0));
            continue;
        }
        if (t != 0 && lane == 0) st_relaxed_gpu_u64(&r.flb_status[t], lb_pack(run, CC_LB_AGG, cnt));
        cc_fused_lookback(r.flb_status, run, t, lane, true, &excl);
        if (lane == 0) st_relaxed_gpu_u64(&r.flb_status[t], lb_pack(run, CC_LB_INC, excl + cnt));
        if ((mask >> lane) & 1u) r.D[excl + __popc(mask & ((1u << lane) - 1u))] = (u32)(p0 + lane);
        if (last && lane == 0)              // every earlier tile has published its count: k is final
            cc_plan_checkpoint(r, log, mode, epoch, excl + cnt, ((mask >> (np - 1)) & 1u) != 0, inline_ok);
        if (!inline_ok) continue;
        // ---- a3 + a5: this warp gathers its own dirty pages (one read -> log payload, shadow, CRC) ----
        u32 m = mask, i = excl;
        while (m) {
            const u32 pl = (u32)__ffs(m) - 1u;
            m &= m - 1;
            const u64 p = p0 + pl;
            const u64 plen = page_len_dev(r, p);
            const uint4* src = reinterpret_cast<const uint4*>(r.base + p * (u64)P);
            uint4* dsh = reinterpret_cast<uint4*>(r.shadow + p * (u64)P);
            u8* rec = log->buf + W0 + (u64)i * rec_stride;
            uint4* dlog = reinterpret_cast<uint4*>(rec + CC_RECORD_HEADER_BYTES);
            const u32 nvec = (u32)(plen >> 4);
            u32 crc = 0;
            for (u32 v0 = 0; v0 < nvec; v0 += CC_SEG_VECS) {
                uint4 v[U];
                u32 nv = nvec - v0;
                if (nv >= CC_SEG_VECS) {
                    nv = CC_SEG_VECS;
#pragma unroll
                    for (int u = 0; u < U; u++) v[u] = ld_v4(src + v0 + lane + 32 * u);
#pragma unroll
                    for (int u = 0; u < U; u++) st_stream(dlog + v0 + lane + 32 * u, v[u]);
                    if (has_shadow) {
#pragma unroll
                        for (int u = 0; u < U; u++) st_stream(dsh + v0 + lane + 32 * u, v[u]);
                    }
                    if (v0) crc = cc_warp_mul_seg(crc, pow_lane, lane);
                } else {
#pragma unroll
                    for (int u = 0; u < U; u++) {
                        const u32 q = lane + 32 * u;
                        if (q < nv) {
                            v[u] = ld_v4(src + v0 + q);
                            st_stream(dlog + v0 + q, v[u]);
                            if (has_shadow) st_stream(dsh + v0 + q, v[u]);
                        } else {
                            v[u] = make_uint4(0, 0, 0, 0);
                        }
                    }
                    if (v0) crc = gf_mul(crc, gf_xpow_bytes(dev->crc.xp, (u64)nv * 16u));
                }
                crc ^= crc_segment_warp<U>(cs, &dev->crc, v, nv, 0, lane);
            }
            if (lane == 0)
                st_u32x4(rec, r.region_id, (u32)p, (u32)plen, crc_finalize(crc, plen == P ? r.crc_init_full : r.crc_init_tail));
            i++;
        }
    }
}
