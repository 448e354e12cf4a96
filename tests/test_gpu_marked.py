"""GPU parity: allocator-aware discovery (cc_checkpoint_marked / cc_checkpoint_versions and their worker tasks)
vs oracle.checkpoint_marked / oracle.checkpoint_versions, bit-exact (dirty list, log bytes, shadow, marks,
committed versions).  SURVEY.md 8f #1."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc

pytestmark = pytest.mark.gpu


def _bitmap(n_pages, pages, junk_tail=False):
    bm = np.zeros((n_pages + 31) // 32, dtype=np.uint32)
    for p in pages:
        bm[p >> 5] |= np.uint32(1 << (p & 31))
    if junk_tail and n_pages % 32:
        bm[-1] |= np.uint32((0xFFFFFFFF << (n_pages % 32)) & 0xFFFFFFFF)     # bits beyond n_pages: ignored
    return bm


def _run_marked(cur, shadow0, P, marks_np, flags, cap, region_id=4, epoch=21, pinned=False):
    """One cc_checkpoint_marked against the oracle on the same bytes.  shadow0 None = CC_REG_NO_SHADOW."""
    verify, consume = bool(flags & cc.CC_MARK_VERIFY), bool(flags & cc.CC_MARK_CONSUME)
    cur_h = cur.cpu().numpy()
    sh_h = None if shadow0 is None else shadow0.cpu().numpy().copy()
    om = marks_np.copy()
    olog = np.zeros(cap, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint_marked(cur_h, sh_h, P, region_id, epoch, om, olog, 0, verify=verify, consume=consume)
    ctx = cc.Context()
    if shadow0 is None:
        shadow = ctx.register_region(region_id, cur, P, no_shadow=True)
        assert shadow is None
    else:
        shadow = shadow0.clone()
        ctx.register_region(region_id, cur, P, shadow=shadow, snapshot_now=False)
    glog = torch.zeros(cap, dtype=torch.uint8, pin_memory=True) if pinned else torch.zeros(cap, dtype=torch.uint8, device="cuda")
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(glog, committed)
    gm = torch.from_numpy(marks_np.view(np.int32).copy()).cuda()
    res = cc.Result()
    ctx.checkpoint_marked(region_id, epoch, gm, flags, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.seq_done, r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch) == (1, st, D.size, nb, W, epoch)
    assert ctx.dirty_list(region_id).tolist() == D.tolist()
    assert np.array_equal(glog.cpu().numpy(), olog), "log bytes differ"
    if shadow is not None:
        assert np.array_equal(shadow.cpu().numpy(), sh_h), "shadow differs"
    assert np.array_equal(gm.cpu().numpy().view(np.uint32), om), "marks differ"
    assert int(committed.item()) == W
    assert np.array_equal(cur.cpu().numpy(), cur_h)
    return ctx, r, D, glog, shadow


@pytest.mark.parametrize("P,n_pages,tail", [(16, 7, 0), (64, 70, 48), (4096, 1100, 1024), (4112, 35, 16),
                                            (16384, 67, 4096 + 16), (65536, 40, 65520), (81920, 9, 4096)])
@pytest.mark.parametrize("flags", [0, cc.CC_MARK_VERIFY, cc.CC_MARK_CONSUME, cc.CC_MARK_VERIFY | cc.CC_MARK_CONSUME])
def test_marked_shapes_and_flags(P, n_pages, tail, flags):
    N = (n_pages - 1) * P + (tail or P)
    cur = synth.raw_region(N, 300 + n_pages, "cuda")
    sh = cur.clone()
    rng = np.random.default_rng(P + n_pages + flags)
    dirty = sorted(set(rng.integers(0, n_pages, max(1, n_pages // 4)).tolist()) | {n_pages - 1})
    for p in dirty:
        plen = min(P, N - p * P)
        sh[p * P + int(rng.integers(0, plen))] ^= 1 << int(rng.integers(0, 8))
    # marks: most of the dirty pages (one dirty page deliberately unmarked) plus some clean ones
    marks = sorted((set(dirty) - {dirty[0]}) | set(rng.integers(0, n_pages, max(1, n_pages // 5)).tolist()))
    ctx, r, D, glog, shadow = _run_marked(cur, sh, P, _bitmap(n_pages, marks, junk_tail=True), flags,
                                          n_pages * (16 + P) + 64)
    if flags & cc.CC_MARK_VERIFY:
        assert D.tolist() == sorted(set(marks) & set(dirty))
    else:
        assert D.tolist() == marks
    ctx.shutdown()


def test_marked_verify_all_marked_equals_plain_checkpoint_and_no_shadow_region():
    P, n_pages = 4096, 777
    N = P * n_pages - 2048
    cur = synth.raw_region(N, 31, "cuda")
    sh = cur.clone()
    pages = synth.mutate_byte_flips(sh, P, 0.05, 32)
    bm = _bitmap(n_pages, range(n_pages))
    cap = n_pages * (16 + P) + 64
    ctx, r, D, glog, shadow = _run_marked(cur, sh, P, bm, cc.CC_MARK_VERIFY, cap, region_id=3, epoch=17)
    # the plain scan path on the same inputs gives the same log
    olog = np.zeros(cap, dtype=np.uint8)
    st, D2, nb, W = oracle.checkpoint(cur.cpu().numpy(), sh.cpu().numpy().copy(), P, 3, 17, olog, 0)
    assert D.tolist() == D2.tolist() == pages.tolist() and np.array_equal(glog.cpu().numpy(), olog)
    ctx.shutdown()
    # no-shadow region: trusted marks only; scan-based calls are refused
    ctx, r, D, glog, shadow = _run_marked(cur, None, P, _bitmap(n_pages, pages.tolist()), cc.CC_MARK_CONSUME, cap, pinned=True)
    assert D.tolist() == pages.tolist()
    gm = torch.zeros((n_pages + 31) // 32, dtype=torch.int32, device="cuda")
    with pytest.raises(cc.ConcordiaError) as e:
        ctx.checkpoint_delta(4, 1)
    assert e.value.code == cc.CC_ERR_INVALID
    with pytest.raises(cc.ConcordiaError):
        ctx.scan_only(4)
    with pytest.raises(cc.ConcordiaError):
        ctx.checkpoint_marked(4, 1, gm, cc.CC_MARK_VERIFY)
    with pytest.raises(cc.ConcordiaError):
        ctx.checkpoint_marked(4, 1, gm, 8)           # unknown flag
    with pytest.raises(cc.ConcordiaError):
        ctx.checkpoint_marked(99, 1, gm, 0)          # unknown region
    # apply onto a no-shadow region works (only the live pages are written)
    ctx.apply_attach(4096)
    old = synth.raw_region(N, 99, "cuda")
    cur_new = cur.clone()
    cur.copy_(old)
    res = cc.Result()
    ctx.apply_log(glog, int(r.bytes), res)
    torch.cuda.synchronize()
    rr = res.read()
    assert (rr.status, rr.n_dirty, rr.bytes) == (0, len(D), r.bytes)
    exp = old.cpu().numpy().copy()
    for p in D.tolist():
        exp[p * P:(p + 1) * P] = cur_new.cpu().numpy()[p * P:(p + 1) * P]
    assert np.array_equal(cur.cpu().numpy(), exp)
    ctx.shutdown()


def test_marked_empty_log_full_and_chaining():
    P, n_pages = 4096, 300
    cur = synth.raw_region(P * n_pages, 41, "cuda")
    ctx = cc.Context()
    sh = ctx.register_region(1, cur, P)
    marks = [0, 1, 2, 100, 299]
    need = len(marks) * (16 + P) + 32
    log = torch.zeros(2 * need - 1, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    res = cc.Result()
    # no marks: nothing appended
    gm = torch.zeros((n_pages + 31) // 32, dtype=torch.int32, device="cuda")
    ctx.checkpoint_marked(1, 1, gm, cc.CC_MARK_CONSUME, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (0, 0, 0, 0) and not log.any()
    # first epoch fits, second does not (all-or-nothing; marks and shadow stay), after a reset it does
    host_cur = cur.cpu().numpy()
    host_sh = host_cur.copy()
    olog = np.zeros(log.numel(), dtype=np.uint8)
    bm = _bitmap(n_pages, marks)
    gm = torch.from_numpy(bm.view(np.int32).copy()).cuda()
    res.clear()
    ctx.checkpoint_marked(1, 2, gm, 0, res)
    torch.cuda.synchronize()
    st, D, nb, W = oracle.checkpoint_marked(host_cur, host_sh, P, 1, 2, bm, olog, 0)
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (0, 5, need, need) == (st, D.size, nb, W)
    cur[5 * P + 7] ^= 3
    host_cur = cur.cpu().numpy()
    sh_before = sh.clone()
    res.clear()
    ctx.checkpoint_marked(1, 3, gm, cc.CC_MARK_CONSUME, res)
    torch.cuda.synchronize()
    r = res.read()
    st, D, nb, W2 = oracle.checkpoint_marked(host_cur, host_sh, P, 1, 3, bm, olog, W, consume=True)
    assert st == oracle.ORC_ERR_LOG_FULL
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (cc.CC_ERR_LOG_FULL, 5, 0, need)
    assert np.array_equal(gm.cpu().numpy().view(np.uint32), bm) and torch.equal(sh, sh_before)
    assert np.array_equal(log.cpu().numpy(), olog)
    ctx.log_reset()
    res.clear()
    ctx.checkpoint_marked(1, 3, gm, cc.CC_MARK_CONSUME, res)
    torch.cuda.synchronize()
    r = res.read()
    st, D, nb, W3 = oracle.checkpoint_marked(host_cur, host_sh, P, 1, 3, bm, olog, 0, consume=True)
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (0, 5, need, need) == (st, D.size, nb, W3)
    assert not gm.any() and not bm.any() and np.array_equal(log.cpu().numpy(), olog)
    # the unmarked dirty page 5 is still found by the transparent diff afterwards
    res.clear()
    ctx.log_reset()
    ctx.checkpoint_delta(1, 4, res)
    torch.cuda.synchronize()
    assert res.read().n_dirty == 1 and ctx.dirty_list(1).tolist() == [5]
    ctx.shutdown()


def test_versions_parity_and_advance():
    P, n_pages = 16384, 211
    N = P * n_pages - 4096
    cur = synth.raw_region(N, 51, "cuda")
    host_cur = cur.cpu().numpy()
    rng = np.random.default_rng(5)
    ver = rng.integers(0, 1 << 62, n_pages, dtype=np.uint64)
    com = ver.copy()
    bumped = sorted(set(rng.integers(0, n_pages, 40).tolist()) | {0, n_pages - 1})
    for p in bumped:
        ver[p] += np.uint64(1)
    ver[bumped[3]] = 0                                   # "different", not "greater"
    cap = n_pages * (16 + P) + 64
    ctx = cc.Context()
    ctx.register_region(2, cur, P, no_shadow=True)
    log = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    small = torch.zeros(1000, dtype=torch.uint8, device="cuda")
    gver = torch.from_numpy(ver.view(np.int64).copy()).cuda()
    gcom = torch.from_numpy(com.view(np.int64).copy()).cuda()
    res = cc.Result()
    # log full first: committed[] must not move
    ctx.log_attach(small)
    ctx.checkpoint_versions(2, 9, gver, gcom, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes) == (cc.CC_ERR_LOG_FULL, len(bumped), 0)
    assert np.array_equal(gcom.cpu().numpy().view(np.uint64), com) and not small.any()
    ctx.log_attach(log)
    olog = np.zeros(cap, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint_versions(host_cur, None, P, 2, 9, ver, com, olog, 0)
    res.clear()
    ctx.checkpoint_versions(2, 9, gver, gcom, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (st, D.size, nb, W) and D.tolist() == bumped
    assert ctx.dirty_list(2).tolist() == bumped
    assert np.array_equal(log.cpu().numpy(), olog)
    assert np.array_equal(gcom.cpu().numpy().view(np.uint64), com) and np.array_equal(com, ver)
    # nothing bumped since: empty
    res.clear()
    ctx.checkpoint_versions(2, 10, gver, gcom, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (0, 0, 0, W)
    ctx.shutdown()


def test_worker_marked_and_version_tasks_equal_host_launched_and_oracle():
    P, n_pages = 4096, 512
    cur = synth.raw_region(P * n_pages, 61, "cuda")
    # 16 worker blocks: the other SMs stay free for the application's own (torch) kernels while the worker is resident
    ctx = cc.Context(ring_capacity=16, worker_blocks=16, max_lifetime_ns=int(30e9))
    sh = ctx.register_region(1, cur, P)
    log = torch.zeros(1 << 22, dtype=torch.uint8, pin_memory=True)
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(log, committed)
    host_cur = cur.cpu().numpy().copy()
    host_sh = host_cur.copy()
    olog = np.zeros(log.numel(), dtype=np.uint8)
    rng = np.random.default_rng(6)
    n_words = (n_pages + 31) // 32
    gm = torch.zeros(n_words, dtype=torch.int32, device="cuda")
    ver = np.zeros(n_pages, dtype=np.uint64)
    com = ver.copy()
    gver = torch.zeros(n_pages, dtype=torch.int64, device="cuda")
    gcom = torch.zeros(n_pages, dtype=torch.int64, device="cuda")
    W = 0
    ctx.worker_start()
    try:
        for task in range(6):
            pages = sorted(set(rng.integers(0, n_pages, 9).tolist()))
            for p in pages:                                   # the "application" writes and marks
                off = p * P + int(rng.integers(0, P))
                host_cur[off] ^= 0x11
                cur[off] ^= 0x11
            torch.cuda.current_stream().synchronize()     # never a device-wide sync under the resident worker
            if task % 2 == 0:
                flags = [0, cc.CC_MARK_VERIFY | cc.CC_MARK_CONSUME, cc.CC_MARK_CONSUME][task // 2]
                marks = sorted(set(pages) | {3, 500})
                bm = _bitmap(n_pages, marks)
                gm.copy_(torch.from_numpy(bm.view(np.int32).copy()))
                torch.cuda.current_stream().synchronize()
                s = ctx.submit(cc.CC_TASK_MARKED_CKPT, region_id=1, epoch=task, arg0=gm.data_ptr(), arg1=flags)
                st, D, nb, W = oracle.checkpoint_marked(host_cur, host_sh, P, 1, task, bm, olog, W,
                                                        verify=bool(flags & 1), consume=bool(flags & 2))
                r = ctx.wait(s, 10.0)
                assert np.array_equal(gm.cpu().numpy().view(np.uint32), bm)
            else:
                for p in pages:
                    ver[p] += np.uint64(task)
                gver.copy_(torch.from_numpy(ver.view(np.int64).copy()))
                torch.cuda.current_stream().synchronize()
                s = ctx.submit(cc.CC_TASK_VERSION_CKPT, region_id=1, epoch=task, arg0=gver.data_ptr(), arg1=gcom.data_ptr())
                st, D, nb, W = oracle.checkpoint_versions(host_cur, host_sh, P, 1, task, ver, com, olog, W)
                r = ctx.wait(s, 10.0)
                assert np.array_equal(gcom.cpu().numpy().view(np.uint64), com)
            assert (r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch) == (st, D.size, nb, W, task), r.as_dict()
        assert int(committed.item()) == W and np.array_equal(log.numpy(), olog)
        # bad arguments are refused per task, the worker keeps running
        s = ctx.submit(cc.CC_TASK_MARKED_CKPT, region_id=1, epoch=1, arg0=0, arg1=0)
        assert ctx.wait(s, 10.0).status == cc.CC_ERR_INVALID
        assert ctx.worker_alive()
    finally:
        ctx.worker_stop()
    torch.cuda.synchronize()
    assert np.array_equal(sh.cpu().numpy(), host_sh)
    ctx.shutdown()


def test_c2_allocator_bitmap_full_size_cost_is_dirty_bytes_only():
    """BASELINE.json configs[1] at full size with the block allocator's dirty bitmap: same log as the scan
    path (the marks equal the dirty set), sampled records checked against the oracle's CRC."""
    free, _ = torch.cuda.mem_get_info()
    if free < 20 * 2**30:
        pytest.skip("needs 20 GiB of device memory")
    layers, blocks, seqs, P = 32, 4096, 256, 65536
    cur = synth.kv_cache_region(layers, blocks, 1002, "cuda")
    ctx = cc.Context()
    sh = ctx.register_region(1, cur, P)
    pages = synth.kv_decode_step(cur, layers, blocks, seqs, 1002)
    n_pages = layers * blocks
    k = pages.numel()
    cap = k * (16 + P) + 32
    log_scan = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    log_mark = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    gm = torch.from_numpy(_bitmap(n_pages, pages.tolist()).view(np.int32).copy()).cuda()
    res = cc.Result()
    sh0 = sh.clone()
    ctx.log_attach(log_mark)
    ctx.checkpoint_marked(1, 5, gm, cc.CC_MARK_CONSUME, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes) == (0, k, cap) and not gm.any()
    assert torch.equal(sh, cur)
    sh.copy_(sh0)
    ctx.log_attach(log_scan)
    res.clear()
    ctx.checkpoint_delta(1, 5, res)
    torch.cuda.synchronize()
    assert res.read().n_dirty == k
    assert torch.equal(log_scan, log_mark)
    # sampled records against the oracle
    for i in np.random.default_rng(0).integers(0, k, 16).tolist():
        rec = log_mark[i * (16 + P):(i + 1) * (16 + P)].cpu().numpy()
        hdr = rec[:16].view(np.uint32)
        p = int(pages[i])
        page = cur[p * P:(p + 1) * P].cpu().numpy()
        assert hdr.tolist() == [1, p, P, oracle.crc32c(page)] and np.array_equal(rec[16:], page)
    ctx.shutdown()
