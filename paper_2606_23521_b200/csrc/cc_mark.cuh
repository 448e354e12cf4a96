// cc_mark.cuh -- allocator-aware dirty discovery: instead of diffing the whole
// region against its shadow, take the dirty set from metadata the serving runtime already has
// ("dirty-block/version metadata", L257 "block-table version counters or dirty-block
// bitmaps supplied by the serving runtime; Concordia then copies the marked physical pages",
// L261 "reads allocator dirty metadata", L264 "Allocator version counters are advanced", L266
// "discovery is proportional to the dirty block bitmap").  These phases only FILL the region's
// dirty bitmap; the ordered compaction (a2) and the gather (a3-a5) are the ones of cc_ckpt.cuh.
#pragma once
#include "cc_common.cuh"

// Every discovery phase opens a new compaction run (same bookkeeping as cc_scan_phase).
__device__ __forceinline__ void cc_open_run(const cc_region_dev& r, cc_grid g, bool stamp) {
    if (g.block == 0 && threadIdx.x == 0) {
        if (stamp) r.hdr->t_start_ns = globaltimer_ns();
        r.hdr->ticket = 0;
        r.hdr->run_id = r.hdr->run_id + 1;
    }
}

// bitmap := marks, with the bits at or beyond n_pages masked off (reading #29).
__device__ __forceinline__ void cc_mark_load_phase(const cc_region_dev& r, const u32* marks, cc_grid g) {
    cc_open_run(r, g, true);
    const u64 nw = r.n_words;
    const u32 tail_bits = (u32)(r.n_pages & 31u);
    for (u64 w = (u64)g.block * blockDim.x + threadIdx.x; w < nw; w += (u64)g.nblocks * blockDim.x) {
        u32 v = marks[w];
        if (w == nw - 1 && tail_bits) v &= (1u << tail_bits) - 1u;
        if (v) r.bitmap[w] = v;
    }
}

// bitmap bit p := version[p] != committed[p]; one warp per bitmap word (coalesced 256-byte reads).
__device__ __forceinline__ void cc_mark_versions_phase(const cc_region_dev& r, const u64* version, const u64* committed,
                                                       cc_grid g) {
    cc_open_run(r, g, true);
    const u32 lane = threadIdx.x & 31u;
    for (u64 w = g.warp(); w < r.n_words; w += g.nwarps()) {
        const u64 p = (w << 5) + lane;
        const bool d = (p < r.n_pages) && (version[p] != committed[p]);
        const u32 word = __ballot_sync(0xFFFFFFFFu, d);
        if (lane == 0 && word) r.bitmap[w] = word;
    }
}

// Verified marks: D[0..k) holds the marked pages (a first compaction in scan-only mode); compare
// only those against the shadow, one warp per 4 KiB segment, and set the bit of a page that
// really differs.  A second compaction then yields the dirty list proper.
__device__ __forceinline__ void cc_mark_verify_phase(const cc_region_dev& r, cc_grid g) {
    constexpr int U = 8;
    cc_open_run(r, g, false);
    const u32 lane = threadIdx.x & 31u;
    const u32 k = r.hdr->k;
    const u32 spp = r.spp;
    const u64 n_items = (u64)k * spp;
    for (u64 item = g.warp(); item < n_items; item += g.nwarps()) {
        u32 i, c;
        if (r.spp_shift >= 0) { i = (u32)(item >> r.spp_shift); c = (u32)(item & (spp - 1)); }
        else { i = (u32)(item / spp); c = (u32)(item - (u64)i * spp); }
        const u64 p = r.D[i];
        const u64 plen = page_len_dev(r, p);
        const u64 so = (u64)c * CC_SEG_BYTES;
        if (so >= plen) continue;
        const u64 rem = plen - so;
        const u32 nv = (u32)((rem < CC_SEG_BYTES ? rem : CC_SEG_BYTES) >> 4);
        const uint4* a = reinterpret_cast<const uint4*>(r.base + p * r.page_bytes + so);
        const uint4* b = reinterpret_cast<const uint4*>(r.shadow + p * r.page_bytes + so);
        uint4 va[U], vb[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            const u32 j = lane + 32 * u;
            va[u] = (j < nv) ? ld_stream(a + j) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
            const u32 j = lane + 32 * u;
            vb[u] = (j < nv) ? ld_stream(b + j) : make_uint4(0, 0, 0, 0);
        }
        u32 acc = 0;
#pragma unroll
        for (int u = 0; u < U; u++)
            acc |= (va[u].x ^ vb[u].x) | (va[u].y ^ vb[u].y) | (va[u].z ^ vb[u].z) | (va[u].w ^ vb[u].w);
        if (__any_sync(0xFFFFFFFFu, acc != 0) && lane == 0)
            atomicOr(&r.bitmap[p >> 5], 1u << (p & 31));
    }
}

// After the gather: hand the metadata back (reading #31/#32).  Only when the checkpoint went
// through (status CC_OK; an empty epoch counts): clear the caller's marks (CONSUME) and/or advance
// committed[p] := version[p] for the pages that were logged.  On CC_ERR_LOG_FULL nothing moves.
__device__ __forceinline__ void cc_mark_finish_phase(const cc_region_dev& r, u32* marks_to_clear, const u64* version,
                                                     u64* committed, cc_grid g) {
    const cc_ws_hdr* h = r.hdr;
    if (h->status != CC_OK) return;
    const u64 tid = (u64)g.block * blockDim.x + threadIdx.x, nthr = (u64)g.nblocks * blockDim.x;
    if (marks_to_clear)
        for (u64 w = tid; w < r.n_words; w += nthr)
            if (marks_to_clear[w]) marks_to_clear[w] = 0;
    if (version && committed) {
        const u32 k = h->k_eff;
        for (u64 i = tid; i < k; i += nthr) {
            const u32 p = r.D[i];
            committed[p] = version[p];
        }
    }
}
