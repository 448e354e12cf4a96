"""GPU parity: base snapshot (cc_snapshot_region) and log compactor (cc_compact_log, CC_TASK_SNAPSHOT /
CC_TASK_COMPACT_LOG) vs oracle.snapshot / oracle.compact_log, bit-exact.  SURVEY.md 8f #3."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc

pytestmark = pytest.mark.gpu


# ------------------------------------------------------------------ base snapshot --

@pytest.mark.parametrize("P,n_pages,tail", [(16, 7, 0), (64, 70, 48), (4096, 300, 1024), (4112, 35, 16),
                                            (65536, 20, 65520), (81920, 9, 4096)])
@pytest.mark.parametrize("with_shadow", [True, False])
def test_snapshot_parity(P, n_pages, tail, with_shadow):
    N = (n_pages - 1) * P + (tail or P)
    cur = synth.raw_region(N, 500 + n_pages, "cuda")
    cur_h = cur.cpu().numpy()
    sh_h = np.zeros(N, np.uint8) if with_shadow else None
    cap = n_pages * (16 + P) + 32 + 48
    olog = np.zeros(cap, np.uint8)
    st, k, nb, W = oracle.snapshot(cur_h, sh_h, P, 6, 44, olog, 0)
    ctx = cc.Context()
    if with_shadow:
        shadow = torch.zeros(N, dtype=torch.uint8, device="cuda")
        ctx.register_region(6, cur, P, shadow=shadow, snapshot_now=False)
    else:
        ctx.register_region(6, cur, P, no_shadow=True)
    glog = torch.zeros(cap, dtype=torch.uint8, pin_memory=True) if n_pages % 2 else torch.zeros(cap, dtype=torch.uint8, device="cuda")
    ctx.log_attach(glog)
    res = cc.Result()
    ctx.snapshot_region(6, 44, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch) == (st, k, nb, W, 44) and k == n_pages
    assert np.array_equal(glog.cpu().numpy(), olog)
    if with_shadow:
        assert torch.equal(shadow, cur)
        # the next delta is relative to the snapshot
        res.clear()
        ctx.checkpoint_delta(6, 45, res)
        torch.cuda.synchronize()
        assert res.read().n_dirty == 0
    # log full: nothing appended
    ctx.log_reset()
    small = torch.zeros(nb - 1, dtype=torch.uint8, device="cuda")
    ctx.log_attach(small)
    res.clear()
    ctx.snapshot_region(6, 46, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes) == (cc.CC_ERR_LOG_FULL, n_pages, 0) and not small.any()
    ctx.shutdown()


# ------------------------------------------------------------------ log compactor --

def _build_log(arena_bytes, n_epochs, recs, seed, forced):
    unit = arena_bytes // 8
    eps = synth.recovery_epochs(arena_bytes, n_epochs, recs, seed, forced_repeats=forced)
    cap = sum(e.payloads.numel() + 16 * e.pages.numel() + 32 for e in eps)
    olog = np.zeros(cap, dtype=np.uint8)
    views = {rid: (o8 * unit, s8 * unit, P) for rid, o8, s8, P in synth.C5A_REGIONS}
    W = 0
    for e in eps:
        o, sz, P = views[e.region_id]
        st, W = oracle.write_epoch(olog, W, e.region_id, e.epoch, sz, P, e.pages.numpy(), e.payloads.numpy())
        assert st == 0
    return olog, W, views, sum(e.pages.numel() for e in eps)


def _ctx_with_regions(arena, views, max_records):
    ctx = cc.Context(ring_capacity=8, max_lifetime_ns=int(60e9))
    for rid in sorted(views, reverse=True):                 # registered in DESCENDING id order on purpose
        o, sz, P = views[rid]
        ctx.register_region(rid, arena[o:o + sz], P)
    ctx.apply_attach(max_records)
    return ctx


def _oregions(host, views):
    return [oracle.Region(rid, P, host[o:o + sz]) for rid, (o, sz, P) in views.items()]


def test_compactor_parity_mixed_regions_duplicates_and_replay_equivalence():
    arena_bytes = 64 << 20
    olog, W, views, n_rec = _build_log(arena_bytes, 30, 40, 1005, forced=10)
    arena = synth.raw_region(arena_bytes, 1005, "cuda")
    host = arena.cpu().numpy().copy()
    exp_out = np.zeros(W, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(olog, W, _oregions(host, views), exp_out)
    assert st == 0 and consumed == W and 0 < n_out < n_rec and nb < W
    for pinned_in, pinned_out in ((False, False), (True, True), (True, False)):
        work = arena.clone()
        ctx = _ctx_with_regions(work, views, n_rec + 64)
        lt = torch.from_numpy(olog)
        lt = lt.pin_memory() if pinned_in else lt.cuda()
        out = torch.zeros(W, dtype=torch.uint8, pin_memory=True) if pinned_out else torch.zeros(W, dtype=torch.uint8, device="cuda")
        res = cc.Result()
        ctx.compact_log(lt, W, out, res)
        torch.cuda.synchronize()
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch) == (0, n_out, nb, W, 3), r.as_dict()
        assert np.array_equal(out.cpu().numpy(), exp_out), "compacted log differs from the oracle's"
        assert torch.equal(work, arena), "compaction must not touch the regions"
        # replaying the compacted log == replaying the original (GPU applier, then against the oracle's replay)
        ctx.apply_log(out, nb, res)
        torch.cuda.synchronize()
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes, r.epoch) == (0, n_out, nb, 3)
        h2 = host.copy()
        assert oracle.apply_log(olog, W, _oregions(h2, views))[0] == 0
        assert np.array_equal(work.cpu().numpy(), h2)
        # compacting the compacted log changes nothing (idempotent); a later checkpoint still works on these regions
        out2 = torch.zeros(W, dtype=torch.uint8, device="cuda")
        res.clear()
        ctx.compact_log(out, nb, out2, res)
        torch.cuda.synchronize()
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes) == (0, n_out, nb) and torch.equal(out2.cpu(), out.cpu())
        ctx.shutdown()


def test_compactor_torn_corrupt_capacity_scratch():
    arena_bytes = 16 << 20
    olog, W, views, n_rec = _build_log(arena_bytes, 9, 12, 77, forced=3)
    arena = synth.raw_region(arena_bytes, 77, "cuda")
    host = arena.cpu().numpy()
    ctx = _ctx_with_regions(arena, views, n_rec + 16)
    lt = torch.from_numpy(olog).cuda()
    res = cc.Result()

    def run(log_t, nbytes, out_t):
        res.clear()
        ctx.compact_log(log_t, nbytes, out_t, res)
        torch.cuda.synchronize()
        return res.read()

    # torn at several cuts: the committed prefix is compacted
    for t in (0, 15, 16, W // 3, W // 2 + 5, W - 1, W):
        exp = np.zeros(W, np.uint8)
        st, nb, consumed, n_out = oracle.compact_log(olog, t, _oregions(host, views), exp)
        out = torch.zeros(W, dtype=torch.uint8, device="cuda")
        r = run(lt, t, out)
        assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (st, n_out, nb, consumed), (t, r.as_dict())
        assert np.array_equal(out.cpu().numpy(), exp)
    # corrupt payload bit / corrupt header / corrupt commit: nothing written
    for pos, val in ((40, 0x01), (W // 2, 0x80), (W - 9, 0x01)):
        bad = olog.copy()
        bad[pos] ^= val
        exp = np.zeros(W, np.uint8)
        st, nb, consumed, n_out = oracle.compact_log(bad, W, _oregions(host, views), exp)
        out = torch.zeros(W, dtype=torch.uint8, device="cuda")
        r = run(torch.from_numpy(bad).cuda(), W, out)
        assert st == oracle.ORC_ERR_CORRUPT == cc.CC_ERR_CORRUPT
        assert (r.status, r.bytes, r.n_dirty, r.log_offset_after) == (st, 0, 0, consumed), (pos, r.as_dict())
        assert not out.any()
    # capacity one byte short: LOG_FULL and nothing written; exact: fits
    exp = np.zeros(W, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(olog, W, _oregions(host, views), exp)
    out = torch.zeros(nb - 16, dtype=torch.uint8, device="cuda")
    r = run(lt, W, out)
    assert r.status == cc.CC_ERR_LOG_FULL and r.bytes == 0 and not out.any()
    out = torch.zeros(nb, dtype=torch.uint8, device="cuda")
    r = run(lt, W, out)
    assert (r.status, r.bytes) == (0, nb) and np.array_equal(out.cpu().numpy(), exp[:nb])
    # overlapping buffers are refused; a too small scratch writes nothing
    with pytest.raises(cc.ConcordiaError):
        ctx.compact_log(lt, W, lt[16:], res)
    ctx.apply_attach(8)
    out = torch.zeros(W, dtype=torch.uint8, device="cuda")
    r = run(lt, W, out)
    assert r.status == cc.CC_ERR_SCRATCH and r.bytes == 0 and not out.any()
    # the regions' own checkpoints still work afterwards (bitmaps / tables were left clean)
    ctx.apply_attach(n_rec + 16)
    logbuf = torch.zeros(1 << 20, dtype=torch.uint8, device="cuda")
    ctx.log_attach(logbuf)
    o, sz, P = views[2]
    arena[o + 3 * P + 1] ^= 1
    res.clear()
    ctx.checkpoint_delta(2, 1, res)
    torch.cuda.synchronize()
    assert res.read().n_dirty == 1 and ctx.dirty_list(2).tolist() == [3]
    ctx.shutdown()


def test_worker_snapshot_and_compact_tasks():
    arena_bytes = 16 << 20
    olog, W, views, n_rec = _build_log(arena_bytes, 12, 10, 91, forced=4)
    arena = synth.raw_region(arena_bytes, 91, "cuda")
    host = arena.cpu().numpy().copy()
    ctx = _ctx_with_regions(arena, views, n_rec + 16)
    o3, sz3, P3 = views[3]
    snap_cap = (sz3 // P3) * (16 + P3) + 32
    alog = torch.zeros(snap_cap, dtype=torch.uint8, pin_memory=True)
    ctx.log_attach(alog)
    lt = torch.from_numpy(olog).pin_memory()
    out = torch.zeros(W, dtype=torch.uint8, pin_memory=True)
    exp = np.zeros(W, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(olog, W, _oregions(host, views), exp)
    osnap = np.zeros(snap_cap, np.uint8)
    sst, sk, snb, sW = oracle.snapshot(host[o3:o3 + sz3], None, P3, 3, 9, osnap, 0)
    ctx.worker_start()
    try:
        s1 = ctx.submit(cc.CC_TASK_COMPACT_LOG, arg0=lt.data_ptr(), arg1=W, arg2=out.data_ptr(), arg3=out.numel())
        s2 = ctx.submit(cc.CC_TASK_SNAPSHOT, region_id=3, epoch=9)
        r1 = ctx.wait(s1, 20.0)
        r2 = ctx.wait(s2, 20.0)
    finally:
        ctx.worker_stop()
    assert (r1.status, r1.n_dirty, r1.bytes, r1.log_offset_after, r1.epoch) == (0, n_out, nb, W, 3), r1.as_dict()
    assert np.array_equal(out.numpy(), exp)
    assert (r2.status, r2.n_dirty, r2.bytes, r2.log_offset_after) == (sst, sk, snb, sW)
    assert np.array_equal(alog.numpy(), osnap)
    ctx.shutdown()


def test_c5a_full_log_compaction_10000_records():
    """The 10,000-record recovery log of BASELINE.json configs[4] (284 MB, 8 GiB arena): compacted log == oracle's."""
    free, _ = torch.cuda.mem_get_info()
    if free < 12 * 2**30:
        pytest.skip("needs 12 GiB of device memory")
    arena_bytes = 8 << 30
    olog, W, views, n_rec = _build_log(arena_bytes, 100, 100, 1005, forced=50)
    arena = torch.empty(arena_bytes, dtype=torch.uint8, device="cuda")        # contents irrelevant to compaction
    ctx = _ctx_with_regions(arena, views, n_rec + 128)
    oregs = [oracle.Region(rid, P, np.zeros(sz, np.uint8)) for rid, (o, sz, P) in views.items()]   # only id / page size / size are read
    exp = np.zeros(W, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(olog, W, oregs, exp)
    assert st == 0 and n_out <= n_rec - 50
    lt = torch.from_numpy(olog).cuda()
    out = torch.zeros(W, dtype=torch.uint8, device="cuda")
    res = cc.Result()
    ctx.compact_log(lt, W, out, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (0, n_out, nb, W)
    assert np.array_equal(out.cpu().numpy(), exp)
    ctx.shutdown()
