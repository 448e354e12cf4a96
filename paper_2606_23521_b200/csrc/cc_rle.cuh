// cc_rle.cuh -- run-length records ("Sparse page maps use index-value records;
// contiguous dirty ranges use run-length encoding").  One record per RUN of consecutive dirty pages:
// {region_id, first page, len = bytes of the whole run, crc32c(all payload bytes of the run)} + the run's pages
// back to back; a run never crosses a page index that is a multiple of run_pages; the commit record counts
// records.  run_pages = 1 gives the single-page format byte for byte.
//
// After the usual scan + ordered compaction (D[0..k) ascending):
//   starts   bit i of S := rank i starts a run  (i == 0, or D[i-1]+1 != D[i], or D[i] % run_pages == 0)
//   rank     the same ordered compaction, run over S: Rfirst[j] = first rank of run j, n_runs
//   plan     Rn[i] = run of rank i (one thread per run), sizes, all-or-nothing log-full decision
//   gather   as cc_gather_items, but a page's bytes go to W + 16*(j+1) + i*P (j = its run, i = its rank: only
//            the region's last page can be short, and it is last) and its CRC contribution is aligned to the end
//            of the RUN; a page's segments combine into the page's word as before, finished pages combine into
//            the run's word, the last page of a run writes the run's header.
#pragma once
#include "cc_common.cuh"
#include "cc_crc.cuh"
#include "cc_ckpt.cuh"

__device__ __forceinline__ void cc_rle_starts_phase(const cc_region_dev& r, u32 run_pages, cc_grid g) {
    if (g.block == 0 && threadIdx.x == 0) {
        r.hdr2->ticket = 0;
        r.hdr2->run_id = r.hdr2->run_id + 1;
    }
    const u32 lane = threadIdx.x & 31u;
    const u32 k = r.hdr->k;
    const u32 nw = (k + 31u) >> 5;
    for (u32 w = g.warp(); w < nw; w += g.nwarps()) {
        const u32 i = (w << 5) + lane;
        bool start = false;
        if (i < k) {
            const u32 p = r.D[i];
            start = (i == 0) || (r.D[i - 1] + 1u != p) || (p % run_pages == 0);
        }
        const u32 word = __ballot_sync(0xFFFFFFFFu, start);
        if (lane == 0 && word) r.S[w] = word;
    }
}

// The ranking pass sees the dirty RANKS as its "pages": S is its bitmap, Rfirst its output list.
__device__ __forceinline__ void cc_rle_rank_phase(const cc_region_dev& r, const cc_log_dev* log) {
    const u32 k = r.hdr->k;
    if (k == 0) return;
    cc_region_dev v = r;
    v.bitmap = r.S;
    v.D = r.Rfirst;
    v.n_pages = k;
    v.n_words = (k + 31u) >> 5;
    v.hdr = r.hdr2;
    v.lb_status = r.lb2;
    cc_compact_phase(v, log, CC_MODE_SCAN_ONLY, 0, nullptr);
}

__device__ __forceinline__ void cc_rle_plan_phase(const cc_region_dev& r, const cc_log_dev* log, u64 epoch, cc_grid g) {
    cc_ws_hdr* h = r.hdr;
    const u32 k = h->k;
    const u32 n_runs = k ? r.hdr2->k : 0u;
    for (u64 j = (u64)g.block * blockDim.x + threadIdx.x; j < n_runs; j += (u64)g.nblocks * blockDim.x) {
        const u32 first = r.Rfirst[j];
        const u32 next = (j + 1 < n_runs) ? r.Rfirst[j + 1] : k;
        for (u32 i = first; i < next; i++) r.Rn[i] = (u32)j;
    }
    if (g.block == 0 && threadIdx.x == 0) {
        if (k) r.Rfirst[n_runs] = k;            // sentinel (read by the gather of the last run)
        h->epoch = epoch;
        u64 need = (u64)n_runs * CC_RECORD_HEADER_BYTES + (u64)k * r.page_bytes + CC_COMMIT_RECORD_BYTES;
        if (k && r.D[k - 1] == (u32)(r.n_pages - 1)) need -= (u64)r.page_bytes - page_len_dev(r, r.n_pages - 1);
        const u64 W = log->W;
        int32_t st = CC_OK;
        u32 k_eff = 0;
        if (k != 0) {
            if (log->buf == nullptr || W + need > log->capacity) st = CC_ERR_LOG_FULL;
            else k_eff = k;
        }
        h->k_eff = k_eff;
        h->commit_k = n_runs;
        h->n_runs = n_runs;
        h->status = st;
        h->W_start = W;
        h->need = k_eff ? need : 0;
        h->gather_done = 0;
        h->inline_done = 0;
        __threadfence();
    }
}

// Items first, first + step, ... of the k_eff * spp (dirty rank, segment) items.  cs must hold the CRC tables.
__device__ __forceinline__ void cc_rle_gather_items(const cc_region_dev& r, cc_dev* dev, cc_crc_smem* cs, u64 first_item, u64 step) {
    constexpr int U = 8;
    cc_ws_hdr* h = r.hdr;
    cc_log_dev* log = &dev->log;
    const u32 k_eff = h->k_eff;
    const u32 lane = threadIdx.x & 31u;
    const u32 P = r.page_bytes;
    const u64 W0 = h->W_start;
    const u32 spp = r.spp;
    const u64 n_items = (u64)k_eff * spp;
    const bool has_shadow = r.shadow != nullptr;
    for (u64 item = first_item; item < n_items; item += step) {
        u32 i, c;
        if (r.spp_shift >= 0) { i = (u32)(item >> r.spp_shift); c = (u32)(item & (spp - 1)); }
        else { i = (u32)(item / spp); c = (u32)(item - (u64)i * spp); }
        const u32 p = r.D[i];
        const u64 plen = page_len_dev(r, p);
        const u64 so = (u64)c * CC_SEG_BYTES;
        if (so >= plen) continue;
        const u64 rem = plen - so;
        const u32 seg_len = (u32)(rem < CC_SEG_BYTES ? rem : CC_SEG_BYTES);
        const u32 nv = seg_len >> 4;
        const u32 nseg = (u32)((plen + CC_SEG_BYTES - 1) / CC_SEG_BYTES);
        // the run this page belongs to
        const u32 j = r.Rn[i];
        const u32 rf = r.Rfirst[j];
        const u32 m = r.Rfirst[j + 1] - rf;
        const u32 p_first = p - (i - rf), p_last = p_first + m - 1;
        const u64 run_bytes = (u64)(m - 1) * P + page_len_dev(r, p_last);
        const u64 pos = (u64)(i - rf) * P + so;
        const u64 after = run_bytes - pos - seg_len;
        const u64 src_off = (u64)p * P + so;
        const uint4* src = reinterpret_cast<const uint4*>(r.base + src_off);
        uint4* dsh = reinterpret_cast<uint4*>(r.shadow + src_off);
        u8* rec = log->buf + W0 + (u64)j * CC_RECORD_HEADER_BYTES + (u64)rf * P;
        uint4* dlog = reinterpret_cast<uint4*>(rec + CC_RECORD_HEADER_BYTES + pos);
        uint4 v[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            const u32 q = lane + 32 * u;
            if (q < nv) {
                v[u] = ld_stream(src + q);
                st_stream(dlog + q, v[u]);
                if (has_shadow) st_stream(dsh + q, v[u]);
            } else {
                v[u] = make_uint4(0, 0, 0, 0);
            }
        }
        const u32 contrib = crc_segment_warp<U>(cs, &dev->crc, v, nv, after, lane);
        if (lane == 0) {
            u32 acc = 0;
            if (crc_record_combine(&r.rec_state[i], nseg, c, contrib, &acc)) {        // the page is complete
                bool finish = (m == 1);
                if (!finish) {
                    u32* w = reinterpret_cast<u32*>(&r.run_state[j]);
                    atomicXor(w, acc);
                    __threadfence();
                    finish = atomicAdd(w + 1, 1u) == m - 1;                              // the run is complete
                    if (finish) {
                        __threadfence();
                        acc = atomicExch(w, 0u);
                        w[1] = 0;
                    }
                }
                if (finish) {
                    u32 it;
                    if (run_bytes == P) it = r.crc_init_full;
                    else if (m == 1) it = r.crc_init_tail;
                    else it = gf_mul(0xFFFFFFFFu, gf_xpow_bytes(dev->crc.xp, run_bytes));
                    st_u32x4(rec, r.region_id, p_first, (u32)run_bytes, crc_finalize(acc, it));
                }
            }
        }
    }
}

__device__ __forceinline__ void cc_rle_gather_phase(const cc_region_dev& r, cc_dev* dev, cc_crc_smem* cs, cc_grid g,
                                                    cc_result* out, u32 kind, bool init_tables) {
    const cc_ws_hdr* h = r.hdr;
    const u32 k_eff = h->k_eff;
    if (k_eff != 0 && (u64)g.block * (blockDim.x >> 5) < (u64)k_eff * r.spp) {
        if (init_tables) cc_crc_smem_init(cs, &dev->crc);
        cc_rle_gather_items(r, dev, cs, g.warp(), g.nwarps());
    }
    cc_gather_complete(r, dev, g, out, kind, (u64)k_eff * r.spp);
}
