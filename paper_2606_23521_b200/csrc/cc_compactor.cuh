// cc_compactor.cuh -- log compactor ("periodic compaction rewrites the log
// into a smaller base snapshot plus recent deltas", L87, L221, L266 "bounding replay time").
//
// Input: a log (device or pinned host).  It is parsed and validated by the applier's own phases
// (cc_apply.cuh: same torn / corrupt rules).  Then, instead of scattering into the regions:
//   mark     latest[page] = last committed record of the page (atomicMax, as in the applier) and the
//            page's bit in its region's dirty bitmap
//   rank     the ordered compaction of cc_ckpt.cuh over every region's bitmap -> ascending page list
//   plan     one thread: regions in ascending region_id order get their output offsets; all-or-nothing
//            capacity check
//   copy     warp per 4 KiB segment: surviving page -> single-page record at its final place in the output; the
//            header of a page that came from a single-page record is that validated record's, a page cut out of
//            a run record gets its own CRC32C;
//            one commit record per region with the epoch number of the last input epoch that touched it
//   cleanup  latest[] back to zero; result
// A failed check (CC_ERR_CORRUPT) or a too small scratch writes nothing: compaction must not launder a
// damaged log.  A torn tail holds no committed data and is dropped.
#pragma once
#include "cc_common.cuh"
#include "cc_ckpt.cuh"
#include "cc_apply.cuh"

__device__ __forceinline__ bool cc_compactor_ok(const cc_dev* dev) { return dev->apply.status == CC_OK; }

__device__ __forceinline__ void cc_compactor_mark_phase(cc_dev* dev, const cc_apply_tabs& T, cc_grid g) {
    if (g.block == 0 && threadIdx.x < CC_MAX_REGIONS && dev->region_used[threadIdx.x]) {
        cc_ws_hdr* h = dev->regions[threadIdx.x].hdr;       // open a compaction run on every region
        h->ticket = 0;
        h->run_id = h->run_id + 1;
    }
    if (!cc_compactor_ok(dev)) return;
    const u32 n = dev->apply.n_commit_recs;
    for (u32 i = g.block * blockDim.x + threadIdx.x; i < n; i += g.nblocks * blockDim.x) {
        const cc_rec rec = T.recs[i];
        const cc_region_dev& r = dev->regions[rec.slot];
        const u32 m = cc_rec_pages(r, rec.len);              // a run record covers m consecutive pages
        for (u32 q = 0; q < m; q++) {
            const u32 p = rec.page_idx + q;
            atomicMax(&r.latest[p], i + 1);
            atomicOr(&r.bitmap[p >> 5], 1u << (p & 31));
        }
    }
}

__device__ __forceinline__ void cc_compactor_rank_phase(cc_dev* dev) {
    for (int s = 0; s < CC_MAX_REGIONS; s++)
        if (dev->region_used[s]) cc_compact_phase(dev->regions[s], &dev->log, CC_MODE_SCAN_ONLY, 0, nullptr);
}

// One block of at least CC_MAX_REGIONS threads (one per region slot).  hdr->W_start of every region := its
// offset in the output; hdr->need := its bytes.  Regions are ranked by id in parallel; the only sequential
// part is the running offset over <= 64 sizes held in shared memory.
__device__ __forceinline__ void cc_compactor_plan_phase(cc_dev* dev, u64 out_capacity) {
    __shared__ u32 s_id[CC_MAX_REGIONS], s_order[CC_MAX_REGIONS], s_k[CC_MAX_REGIONS], s_n;
    __shared__ u64 s_need[CC_MAX_REGIONS], s_off[CC_MAX_REGIONS];
    cc_compactor_state* C = &dev->compactor;
    const u32 t = threadIdx.x;
    const bool ok = cc_compactor_ok(dev);
    const bool part = ok && t < CC_MAX_REGIONS && dev->region_used[t];
    if (t < CC_MAX_REGIONS) s_id[t] = part ? dev->regions[t].region_id : 0xFFFFFFFFu;
    if (t == 0) s_n = 0;
    __syncthreads();
    if (part) {
        const cc_region_dev& r = dev->regions[t];
        u32 rank = 0;
        for (u32 q = 0; q < CC_MAX_REGIONS; q++) rank += (s_id[q] < s_id[t]) ? 1u : 0u;
        s_order[rank] = t;
        atomicAdd(&s_n, 1u);
        const u32 k = r.hdr->k;
        u64 need = 0;
        if (k) {
            need = (u64)k * ((u64)r.page_bytes + CC_RECORD_HEADER_BYTES) + CC_COMMIT_RECORD_BYTES;
            if (r.D[k - 1] == (u32)(r.n_pages - 1)) need -= (u64)r.page_bytes - page_len_dev(r, r.n_pages - 1);
        }
        s_k[t] = k;
        s_need[t] = need;
    }
    __syncthreads();
    if (t == 0) {
        u64 o = 0, n_out = 0;
        u32 n_reg = 0;
        for (u32 i = 0; i < s_n; i++) {
            const u32 q = s_order[i];
            s_off[q] = o;
            o += s_need[q];
            n_out += s_k[q];
            n_reg += s_k[q] ? 1u : 0u;
        }
        int32_t st = dev->apply.status;
        if (st == CC_OK && o > out_capacity) st = CC_ERR_LOG_FULL;
        C->status = st;
        C->bytes_out = st == CC_OK ? o : 0;
        C->n_out = st == CC_OK ? n_out : 0;
        C->n_regions_out = st == CC_OK ? n_reg : 0;
    }
    __syncthreads();
    if (part) {
        dev->regions[t].hdr->W_start = s_off[t];
        dev->regions[t].hdr->need = s_need[t];
    }
    __threadfence();
}

// cs must hold the CRC tables (a page cut out of a run record needs its own CRC).
__device__ __forceinline__ void cc_compactor_copy_phase(cc_dev* dev, const cc_apply_tabs& T, cc_crc_smem* cs, const u8* in, u8* out,
                                                        cc_grid g) {
    constexpr int U = 8;
    if (dev->compactor.status != CC_OK) return;
    const u32 lane = threadIdx.x & 31u;
    for (int s = 0; s < CC_MAX_REGIONS; s++) {
        if (!dev->region_used[s]) continue;
        const cc_region_dev& r = dev->regions[s];
        const u32 k = r.hdr->k;
        if (k == 0) continue;
        u8* base = out + r.hdr->W_start;
        const u64 rec_stride = (u64)r.page_bytes + CC_RECORD_HEADER_BYTES;
        const u32 spp = r.spp;
        const u64 n_items = (u64)k * spp;
        for (u64 item = g.warp(); item < n_items; item += g.nwarps()) {
            u32 i, c;
            if (r.spp_shift >= 0) { i = (u32)(item >> r.spp_shift); c = (u32)(item & (spp - 1)); }
            else { i = (u32)(item / spp); c = (u32)(item - (u64)i * spp); }
            const u32 p = r.D[i];
            const cc_rec rec = T.recs[r.latest[p] - 1];
            const u64 plen = page_len_dev(r, p);
            const u64 so = (u64)c * CC_SEG_BYTES;
            if (so >= plen) continue;
            const u64 rem = plen - so;
            const u32 seg_len = (u32)(rem < CC_SEG_BYTES ? rem : CC_SEG_BYTES);
            const u32 nv = seg_len >> 4;
            // the page's bytes inside its (possibly multi-page) record
            const uint4* src = reinterpret_cast<const uint4*>(in + rec.off + CC_RECORD_HEADER_BYTES +
                                                              (u64)(p - rec.page_idx) * r.page_bytes + so);
            u8* orec = base + (u64)i * rec_stride;
            uint4* dst = reinterpret_cast<uint4*>(orec + CC_RECORD_HEADER_BYTES + so);
            uint4 v[U];
#pragma unroll
            for (int u = 0; u < U; u++) {
                const u32 j = lane + 32 * u;
                v[u] = (j < nv) ? ld_v4(src + j) : make_uint4(0, 0, 0, 0);
            }
#pragma unroll
            for (int u = 0; u < U; u++) {
                const u32 j = lane + 32 * u;
                if (j < nv) st_stream(dst + j, v[u]);
            }
            if ((u64)rec.len == plen) {                     // single-page record: its validated header is the page's
                if (c == 0 && lane == 0) st_u32x4(orec, r.region_id, p, rec.len, rec.crc);
            } else {                                        // cut out of a run: the page gets its own CRC
                const u32 nseg = (u32)((plen + CC_SEG_BYTES - 1) / CC_SEG_BYTES);
                const u32 contrib = crc_segment_warp<U>(cs, &dev->crc, v, nv, rem - seg_len, lane);
                if (lane == 0) {
                    u32 acc = 0;
                    if (crc_record_combine(&r.rec_state[i], nseg, c, contrib, &acc))
                        st_u32x4(orec, r.region_id, p, (u32)plen,
                                 crc_finalize(acc, plen == r.page_bytes ? r.crc_init_full : r.crc_init_tail));
                }
            }
        }
        if (g.block == 0 && threadIdx.x == 0) {             // the region's commit record
            u8* cm = base + r.hdr->need - CC_COMMIT_RECORD_BYTES;
            const u32 le = dev->compactor.region_last[s];        // last input epoch that touched the region
            const u64 epoch = le ? T.epochs[le - 1].epoch_no : 0ull;
            u32 pay[4] = {(u32)epoch, (u32)(epoch >> 32), r.region_id, k};
            const u32 crc = crc_serial(&dev->crc, reinterpret_cast<const u8*>(pay), 16);
            st_u32x4(cm + 16, pay[0], pay[1], pay[2], pay[3]);
            st_u32x4(cm, CC_COMMIT_ID, CC_COMMIT_ID, 16u, crc);
        }
    }
}

// latest[] back to zero (the rank phase already cleared the bitmaps); result.
__device__ __forceinline__ void cc_compactor_cleanup_phase(cc_dev* dev, const cc_apply_tabs& T, cc_grid g, cc_result* out,
                                                           u32 kind) {
    cc_apply_state* A = &dev->apply;
    if (A->status == CC_OK) {
        const u32 n = A->n_commit_recs;
        for (u32 i = g.block * blockDim.x + threadIdx.x; i < n; i += g.nblocks * blockDim.x) {
            const cc_rec rec = T.recs[i];
            const cc_region_dev& r = dev->regions[rec.slot];
            const u32 m = cc_rec_pages(r, rec.len);
            for (u32 q = 0; q < m; q++) r.latest[rec.page_idx + q] = 0;
        }
    }
    if (g.block == 0 && threadIdx.x == 0 && out) {
        const cc_compactor_state* C = &dev->compactor;
        out->n_dirty = C->n_out;
        out->bytes = C->bytes_out;
        out->log_offset_after = A->consumed;
        out->epoch = C->n_regions_out;
        out->status = C->status;
        out->flags = kind;
        out->t_start_ns = A->t_start_ns;
        out->t_end_ns = globaltimer_ns();
        __threadfence_system();
        st_release_sys_u64(&out->seq_done, 1ull);
    }
}
