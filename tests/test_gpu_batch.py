"""GPU parity: one boundary, all regions (cc_checkpoint_all, CC_TASK_CKPT_ALL) vs oracle.checkpoint_all, bit-exact.
SURVEY.md 8f #4."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc

pytestmark = pytest.mark.gpu

SPECS = [(9, 65536, 65536 * 40 - 4096), (2, 4096, 4096 * 700), (5, 16384, 16384 * 130), (7, 4096, 4096 * 64),
         (30, 64, 64 * 999 - 16), (11, 81920, 81920 * 7)]          # ids unsorted; region 7 gets no shadow


def _setup(seed, log_cap, pinned=False, **ctx_kw):
    rng = np.random.default_rng(seed)
    ctx = cc.Context(**ctx_kw)
    regs, tensors = [], {}
    for rid, P, N in SPECS:
        cur = synth.raw_region(N, seed * 100 + rid, "cuda")
        if rid == 7:
            ctx.register_region(rid, cur, P, no_shadow=True)
            regs.append(oracle.Region(rid, P, cur.cpu().numpy().copy(), None))
            tensors[rid] = (cur, None)
        else:
            sh = ctx.register_region(rid, cur, P)
            h = cur.cpu().numpy().copy()
            regs.append(oracle.Region(rid, P, h, h.copy()))
            tensors[rid] = (cur, sh)
    log = torch.zeros(log_cap, dtype=torch.uint8, pin_memory=True) if pinned else torch.zeros(log_cap, dtype=torch.uint8, device="cuda")
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(log, committed)
    return ctx, regs, tensors, log, committed, rng


def _mutate(regs, tensors, rng, frac=0.05, skip=()):
    for r in regs:
        if r.region_id in skip:
            continue
        N, P = r.base.size, r.page_bytes
        n_pages = (N + P - 1) // P
        cur = tensors[r.region_id][0]
        for p in set(rng.integers(0, n_pages, max(1, int(frac * n_pages))).tolist()) | {n_pages - 1}:
            off = p * P + int(rng.integers(0, min(P, N - p * P)))
            r.base[off] ^= 0x77
            cur[off] ^= 0x77


@pytest.mark.parametrize("pinned", [False, True])
def test_checkpoint_all_equals_the_oracle_sequence(pinned):
    cap = 64 << 20
    ctx, regs, tensors, log, committed, rng = _setup(3, cap, pinned)
    olog = np.zeros(cap, np.uint8)
    W = 0
    res = cc.Result()
    for epoch in range(4):
        if epoch == 2:
            _mutate(regs, tensors, rng, skip=(2, 9, 30))            # some regions clean at this boundary
        elif epoch < 3:
            _mutate(regs, tensors, rng)                              # epoch 3: nothing changed at all
        st, ks, sts, kt, bt, W = oracle.checkpoint_all(regs, 50 + epoch, olog, W)
        res.clear()
        ctx.checkpoint_all(50 + epoch, res)
        torch.cuda.synchronize()
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch) == (st, kt, bt, W, 50 + epoch), r.as_dict()
        assert int(committed.item()) == W
        for i, rg in enumerate(regs):
            if rg.shadow is not None:
                assert ctx.dirty_list(rg.region_id).numel() == ks[i]
    assert np.array_equal(log.cpu().numpy(), olog)
    for rg in regs:
        if rg.shadow is not None:
            assert np.array_equal(tensors[rg.region_id][1].cpu().numpy(), rg.shadow)
    # region 7 (no shadow) was mutated too and never logged
    assert not np.array_equal(tensors[7][0].cpu().numpy(), synth.raw_region(SPECS[3][2], 307, "cuda").cpu().numpy())
    # the batched log replays like any other log
    ctx.apply_attach(20000)
    for rid, (cur, sh) in tensors.items():
        if sh is not None:
            cur.zero_()
    ctx.apply_log(log, W, res)
    torch.cuda.synchronize()
    assert res.read().status == 0
    ctx.shutdown()


def test_checkpoint_all_skips_the_region_that_does_not_fit():
    ctx, regs, tensors, log, committed, rng = _setup(4, 64 << 20)
    _mutate(regs, tensors, rng)
    # sizes of the individual epochs, in ascending id order
    need = {}
    for rg in sorted(regs, key=lambda r: r.region_id):
        if rg.shadow is None:
            continue
        tmp = np.zeros(64 << 20, np.uint8)
        st, D, nb, _ = oracle.checkpoint(rg.base, rg.shadow.copy(), rg.page_bytes, rg.region_id, 1, tmp, 0)
        need[rg.region_id] = nb
    ids = sorted(need)
    cap = need[ids[0]] + need[ids[1]] + need[ids[2]] - 16 + need[ids[3]]     # the third (9) cannot fit, the fourth (11) can
    small = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    ctx.log_attach(small, committed)
    olog = np.zeros(cap, np.uint8)
    st, ks, sts, kt, bt, W = oracle.checkpoint_all(regs, 1, olog, 0)
    assert st == oracle.ORC_ERR_LOG_FULL and sum(1 for s in sts if s) >= 1
    res = cc.Result()
    ctx.checkpoint_all(1, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (cc.CC_ERR_LOG_FULL, kt, bt, W), r.as_dict()
    assert np.array_equal(small.cpu().numpy(), olog) and int(committed.item()) == W
    for rg in regs:
        if rg.shadow is not None:
            assert np.array_equal(tensors[rg.region_id][1].cpu().numpy(), rg.shadow)
    ctx.shutdown()


def test_worker_ckpt_all_task_and_no_regions():
    cap = 32 << 20
    ctx, regs, tensors, log, committed, rng = _setup(5, cap, pinned=True, ring_capacity=8, max_lifetime_ns=int(60e9))
    olog = np.zeros(cap, np.uint8)
    W = 0
    _mutate(regs, tensors, rng)
    torch.cuda.synchronize()
    ctx.worker_start()
    try:
        for epoch in (7, 8):
            st, ks, sts, kt, bt, W = oracle.checkpoint_all(regs, epoch, olog, W)
            s = ctx.submit(cc.CC_TASK_CKPT_ALL, epoch=epoch)
            r = ctx.wait(s, 20.0)
            assert (r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch) == (st, kt, bt, W, epoch), r.as_dict()
    finally:
        ctx.worker_stop()
    assert np.array_equal(log.numpy(), olog) and int(committed.item()) == W
    ctx.shutdown()
    # a context with no shadowed region: the call completes with an empty result
    ctx = cc.Context()
    cur = synth.raw_region(4096 * 8, 1, "cuda")
    ctx.register_region(1, cur, 4096, no_shadow=True)
    ctx.log_attach(torch.zeros(4096, dtype=torch.uint8, device="cuda"))
    res = cc.Result()
    ctx.checkpoint_all(3, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.seq_done, r.status, r.n_dirty, r.bytes) == (1, 0, 0, 0)
    ctx.shutdown()


def _oracle_all_rle(regs, epoch, run_pages, olog, W):
    """reading #37 + #38: the regions that have a shadow, ascending region_id, each as oracle.checkpoint_rle; a region that
    does not fit is skipped whole, the ones after it are still tried; status = the first failure's."""
    st_all, k_tot, b_tot = 0, 0, 0
    for rg in sorted((r for r in regs if r.shadow is not None), key=lambda r: r.region_id):
        st, D, _runs, nb, W2 = oracle.checkpoint_rle(rg.base, rg.shadow, rg.page_bytes, rg.region_id, epoch, run_pages, olog, W)
        k_tot += D.size
        if st == 0:
            b_tot += nb
            W = W2
        elif st_all == 0:
            st_all = st
    return st_all, k_tot, b_tot, W


def _mutate_runs(regs, tensors, rng, skip=()):
    """runs of 1..9 consecutive dirty pages (so that run-length records have something to join)"""
    for r in regs:
        if r.region_id in skip:
            continue
        N, P = r.base.size, r.page_bytes
        n_pages = (N + P - 1) // P
        cur = tensors[r.region_id][0]
        pages = {n_pages - 1}
        for s in rng.integers(0, n_pages, max(1, n_pages // 40)).tolist():
            pages |= set(range(s, min(n_pages, s + int(rng.integers(1, 10)))))
        for p in pages:
            off = p * P + int(rng.integers(0, min(P, N - p * P)))
            r.base[off] ^= 0x31
            cur[off] ^= 0x31


@pytest.mark.parametrize("run_pages", [1, 4, 32, 64])
def test_checkpoint_all_rle_equals_the_oracle_sequence(run_pages):
    """cc_checkpoint_all_rle: run-length records at a multi-region boundary (run_pages <= 32: the single pass per region,
    64: the phases), incl. boundaries where some or all regions are clean; the log replays through the applier."""
    cap = 64 << 20
    ctx, regs, tensors, log, committed, rng = _setup(11 + run_pages, cap)
    start = {rid: t[0].clone() for rid, t in tensors.items()}
    olog = np.zeros(cap, np.uint8)
    W = 0
    res = cc.Result()
    for epoch in range(4):
        if epoch == 2:
            _mutate_runs(regs, tensors, rng, skip=(2, 9, 30))
        elif epoch < 3:
            _mutate_runs(regs, tensors, rng)
        st, kt, bt, W = _oracle_all_rle(regs, 70 + epoch, run_pages, olog, W)
        res.clear()
        ctx.checkpoint_all_rle(70 + epoch, run_pages, res)
        torch.cuda.synchronize()
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch, r.seq_done) == (st, kt, bt, W, 70 + epoch, 1), r.as_dict()
        assert int(committed.item()) == W
    assert np.array_equal(log.cpu().numpy(), olog)
    for rg in regs:
        if rg.shadow is not None:
            assert np.array_equal(tensors[rg.region_id][1].cpu().numpy(), rg.shadow)
    # replay onto the starting state
    final = {rid: t[0].clone() for rid, t in tensors.items()}
    for rid, (cur, sh) in tensors.items():
        if sh is not None:
            cur.copy_(start[rid])
            sh.copy_(start[rid])
    ctx.apply_attach(50000)
    res.clear()
    ctx.apply_log(log, W, res)
    torch.cuda.synchronize()
    assert res.read().status == 0
    for rid, (cur, sh) in tensors.items():
        if sh is not None:
            assert torch.equal(cur, final[rid]) and torch.equal(sh, final[rid])


def test_checkpoint_all_rle_skips_a_region_that_does_not_fit_and_checks_arguments():
    """A middle region whose records do not fit is skipped whole (shadow untouched), the later ones are still logged;
    status = that region's; a retry after a reset logs exactly the skipped region."""
    ctx, regs, tensors, log, committed, rng = _setup(23, 5 << 19)
    _mutate_runs(regs, tensors, rng)
    # make region 9 (64 KiB pages) too big for what is left: dirty every page
    big = next(r for r in regs if r.region_id == 9)
    big.base[::4096] ^= 0x01
    tensors[9][0][::4096] ^= 0x01
    cap = log.numel()
    olog = np.zeros(cap, np.uint8)
    st, kt, bt, W = _oracle_all_rle(regs, 5, 8, olog, 0)
    assert st == cc.CC_ERR_LOG_FULL and W > 0
    res = cc.Result()
    ctx.checkpoint_all_rle(5, 8, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (st, kt, bt, W), r.as_dict()
    assert np.array_equal(log.cpu().numpy(), olog)
    assert np.array_equal(tensors[9][1].cpu().numpy(), big.shadow)             # untouched
    with pytest.raises(cc.ConcordiaError) as e:
        ctx.checkpoint_all_rle(6, 0, res)
    assert e.value.code == cc.CC_ERR_INVALID
    with pytest.raises(cc.ConcordiaError) as e:
        ctx.checkpoint_all_rle(6, 1 << 20, res)                                 # run_pages * 81920 >= 2^32
    assert e.value.code == cc.CC_ERR_INVALID
