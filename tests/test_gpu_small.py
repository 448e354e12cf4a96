"""GPU parity of the small-region path (CC_PATH_SMALL, csrc/cc_small.cuh): one launch, one grid-wide rendezvous, every
block ranks the dirty bitmap by itself.  Bit-exact with the CPU oracle: dirty list, log bytes, shadow, result."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc

pytestmark = pytest.mark.gpu


def _small(ctx, rid, epoch, res):
    res.clear()
    ctx.checkpoint_ex(rid, epoch, res, path=cc.CC_PATH_SMALL)
    torch.cuda.synchronize()
    return res.read()


def _parity(cur, sh0, P, pinned=False, cap=None, rid=3, epoch=17, calls=1):
    N = cur.numel()
    n_pages = (N + P - 1) // P
    cap = cap if cap is not None else n_pages * (16 + P) + 32 + 64
    ctx = cc.Context()
    shadow = sh0.clone()
    ctx.register_region(rid, cur, P, shadow=shadow, snapshot_now=False)
    glog = torch.zeros(cap, dtype=torch.uint8, pin_memory=True) if pinned else torch.zeros(cap, dtype=torch.uint8, device="cuda")
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(glog, committed)
    olog = np.zeros(cap, np.uint8)
    osh = sh0.cpu().numpy().copy()
    st, D, nb, W = oracle.checkpoint(cur.cpu().numpy(), osh, P, rid, epoch, olog, 0)
    res = cc.Result()
    r = _small(ctx, rid, epoch, res)
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch, r.seq_done) == (st, D.size, nb, W, epoch, 1)
    assert ctx.dirty_list(rid).tolist() == D.tolist()
    assert int(committed.item()) == W
    g = glog.cpu().numpy()
    assert np.array_equal(g, olog), "log bytes differ at %s" % np.nonzero(g != olog)[0][:8]
    assert np.array_equal(shadow.cpu().numpy(), osh)
    return ctx, glog, shadow, res, olog, W


@pytest.mark.parametrize("pinned", [False, True])
@pytest.mark.parametrize("P,n_pages,tail", [(16, 7, 0), (64, 9, 48), (256, 33, 0), (4096, 70, 0), (4096, 37, 1024), (4112, 5, 16),
                                            (16384, 19, 4096 + 16), (65536, 6, 0), (65536, 5, 65520), (81920, 4, 4096), (1 << 20, 3, 0),
                                            (4096, 5000, 0), (512, 40000, 256)])
def test_small_path_shapes(P, n_pages, tail, pinned):
    N = (n_pages - 1) * P + (tail or P)
    cur = synth.raw_region(N, 300 + P % 97 + n_pages, "cuda")
    sh = cur.clone()
    rng = np.random.default_rng(P + n_pages)
    for p in sorted(set(rng.integers(0, n_pages, max(1, n_pages // 3)).tolist()) | {0, n_pages - 1}):
        plen = min(P, N - p * P)
        sh[p * P + int(rng.integers(0, plen))] ^= 1 << int(rng.integers(0, 8))
    _parity(cur, sh, P, pinned=pinned)


def test_small_path_nothing_dirty_and_everything_dirty():
    P, N = 4096, 4096 * 129 + 2048
    cur = synth.raw_region(N, 5, "cuda")
    ctx, glog, sh, res, olog, W = _parity(cur, cur.clone(), P)
    assert W == 0 and not glog.any()
    _parity(cur, ~cur, P)


def test_small_path_at_the_page_limit_and_beyond():
    """131,072 pages (4,096 bitmap words) is the most a block ranks by itself; one page more is refused."""
    P = 256
    for n_pages, ok in ((131072, True), (131072 - 31, True), (131073, False)):
        N = n_pages * P
        cur = synth.raw_region(N, 7, "cuda")
        sh = cur.clone()
        rng = np.random.default_rng(n_pages)
        for p in sorted(set(rng.integers(0, n_pages, 3000).tolist()) | {0, 1, 31, 32, n_pages - 2, n_pages - 1}):
            sh[p * P + int(rng.integers(0, P))] ^= 0x40
        if ok:
            _parity(cur, sh, P)
        else:
            ctx = cc.Context()
            ctx.register_region(1, cur, P, shadow=sh, snapshot_now=False)
            ctx.log_attach(torch.zeros(1 << 20, dtype=torch.uint8, device="cuda"))
            with pytest.raises(cc.ConcordiaError) as e:
                ctx.checkpoint_ex(1, 1, cc.Result(), path=cc.CC_PATH_SMALL)
            assert e.value.code == cc.CC_ERR_INVALID


def test_small_path_refuses_other_record_kinds_and_discoveries():
    cur = synth.raw_region(1 << 20, 9, "cuda")
    ctx = cc.Context()
    ctx.register_region(1, cur, 4096)
    ctx.log_attach(torch.zeros(1 << 21, dtype=torch.uint8, device="cuda"))
    for kw in ({"run_pages": 4}, {"discovery": cc.CC_DISC_ALL}):
        with pytest.raises(cc.ConcordiaError) as e:
            ctx.checkpoint_ex(1, 1, cc.Result(), path=cc.CC_PATH_SMALL, **kw)
        assert e.value.code == cc.CC_ERR_INVALID


def test_small_path_log_full_then_retry_and_chained_epochs():
    """All-or-nothing (reading #10): a checkpoint that does not fit appends nothing, leaves the shadow alone and can be
    retried after a reset; consecutive epochs chain their offsets; the bytes equal the oracle's throughout."""
    P, n_pages = 4096, 600
    cur = synth.raw_region(P * n_pages, 11, "cuda")
    old = cur.clone()
    ctx = cc.Context()
    shadow = ctx.register_region(2, cur, P, shadow=old.clone(), snapshot_now=False)
    cap = 40 * (16 + P) + 32
    glog = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    ctx.log_attach(glog)
    host = [cur.cpu().numpy().copy(), old.cpu().numpy().copy()]      # oracle's cur, shadow
    olog = np.zeros(cap, np.uint8)
    res = cc.Result()
    rng = np.random.default_rng(3)
    W = 0
    for epoch, k in enumerate((25, 10, 30, 3), start=1):
        pages = rng.choice(n_pages, k, replace=False)
        for p in pages:
            cur[int(p) * P + int(rng.integers(0, P))] ^= 0x21
        host[0] = cur.cpu().numpy().copy()
        st, D, nb, W_o = oracle.checkpoint(host[0], host[1], P, 2, epoch, olog, W)
        r = _small(ctx, 2, epoch, res)
        assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (st, D.size, nb, W_o)
        assert np.array_equal(glog.cpu().numpy(), olog) and np.array_equal(shadow.cpu().numpy(), host[1])
        if st == cc.CC_ERR_LOG_FULL:
            assert r.bytes == 0 and W_o == W
            ctx.log_reset()
            olog[:] = 0
            glog.zero_()
            st, D, nb, W_o = oracle.checkpoint(host[0], host[1], P, 2, epoch, olog, 0)
            r = _small(ctx, 2, epoch, res)
            assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (st, D.size, nb, W_o) and st == 0
            assert np.array_equal(glog.cpu().numpy(), olog) and np.array_equal(shadow.cpu().numpy(), host[1])
        W = W_o
    assert W > 0


@pytest.mark.parametrize("name", ["c1", "c3"])
def test_small_path_full_configs_one_launch_same_bytes_as_auto(name):
    """BASELINE.json configs[0] and configs[2] at full size through CC_PATH_SMALL (ONE kernel launch) and through
    cc_checkpoint_delta (AUTO: the three chained kernels): same bytes; then applied back onto the old snapshot."""
    if name == "c1":
        P = 4096
        cur = synth.raw_region(64 << 20, 1001, "cuda")
        old = cur.clone()
        pages = synth.mutate_byte_flips(cur, P, 0.01, 1001)
    else:
        P = 65536
        cur = synth.lora_region(32, 1003, "cuda")
        old = cur.clone()
        pages = synth.lora_update(cur, P, 0.05, 1003)
    ctx, glog, shadow, res, olog, W = _parity(cur.view(torch.uint8).view(-1), old.view(torch.uint8).view(-1), P, rid=1, epoch=7)
    assert ctx.dirty_list(1).tolist() == pages.tolist()
    # one launch for the small path ...
    ctx.log_reset()
    shadow.copy_(old.view(torch.uint8).view(-1))
    glog.zero_()
    n0 = ctx.kernel_launches()
    res.clear()
    ctx.checkpoint_ex(1, 7, res, path=cc.CC_PATH_SMALL)
    torch.cuda.synchronize()
    assert ctx.kernel_launches() - n0 == 1
    assert res.read().n_dirty == len(pages) and np.array_equal(glog.cpu().numpy(), olog)
    # ... and the same bytes through cc_checkpoint_delta
    ctx.log_reset()
    shadow.copy_(old.view(torch.uint8).view(-1))
    glog.zero_()
    res.clear()
    ctx.checkpoint_delta(1, 7, res)
    torch.cuda.synchronize()
    assert res.read().n_dirty == len(pages) and np.array_equal(glog.cpu().numpy(), olog)
    # apply onto the old snapshot
    new = cur.clone()
    cur.copy_(old)
    shadow.copy_(old.view(torch.uint8).view(-1))
    ctx.apply_attach(len(pages) + 8)
    res.clear()
    ctx.apply_log(glog, W, res)
    torch.cuda.synchronize()
    assert res.read().status == 0 and torch.equal(cur, new)


def test_small_path_repeated_calls_leave_the_workspace_clean():
    """The bitmap is cleared by the last block of every call: alternate the small path, the phases and the single pass on
    one region with changing dirty sets."""
    P, n_pages = 4096, 3000
    cur = synth.raw_region(P * n_pages, 13, "cuda")
    ctx = cc.Context()
    shadow = ctx.register_region(1, cur, P)
    cap = n_pages * (16 + P) + 32
    glog = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    ctx.log_attach(glog)
    res = cc.Result()
    rng = np.random.default_rng(5)
    for it, path in enumerate([cc.CC_PATH_SMALL, cc.CC_PATH_PHASES, cc.CC_PATH_SMALL, cc.CC_PATH_SINGLE_PASS, cc.CC_PATH_SMALL,
                               cc.CC_PATH_SMALL]):
        pages = sorted(set(rng.integers(0, n_pages, int(rng.integers(1, 200))).tolist()))
        for p in pages:
            cur[p * P + int(rng.integers(0, P))] ^= 0x08
        osh = shadow.cpu().numpy().copy()
        olog = np.zeros(cap, np.uint8)
        st, D, nb, W = oracle.checkpoint(cur.cpu().numpy(), osh, P, 1, it, olog, 0)
        assert D.tolist() == pages
        ctx.log_reset()
        res.clear()
        ctx.checkpoint_ex(1, it, res, path=path)
        torch.cuda.synchronize()
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes) == (st, D.size, nb)
        assert ctx.dirty_list(1).tolist() == pages
        assert np.array_equal(glog.cpu().numpy()[:nb], olog[:nb]) and np.array_equal(shadow.cpu().numpy(), osh)
