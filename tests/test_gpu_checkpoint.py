"""GPU parity: cc_checkpoint_delta vs the CPU oracle, bit-exact (dirty list, log bytes, shadow)."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc
from gpu_util import check_checkpoint_parity, gpu_checkpoint

pytestmark = pytest.mark.gpu


def _region(n, seed):
    return synth.raw_region(n, seed, "cuda")


@pytest.mark.parametrize("P,n_pages,tail", [(16, 7, 0), (64, 9, 48), (256, 33, 0), (4096, 70, 0), (4096, 37, 1024),
                                            (4112, 5, 16), (16384, 19, 4096 + 16), (65536, 6, 0), (65536, 5, 65520),
                                            (81920, 4, 4096), (1 << 20, 3, 0)])
def test_small_shapes(P, n_pages, tail):
    """Sizes that span several tiles and a ragged tail; tiny pages; pages that are not a multiple of 4 KiB."""
    N = (n_pages - 1) * P + (tail or P)
    cur = _region(N, 100 + P % 97 + n_pages)
    sh = cur.clone()
    rng = np.random.default_rng(P + n_pages)
    for p in sorted(set(rng.integers(0, n_pages, max(1, n_pages // 3)).tolist()) | {n_pages - 1}):
        plen = min(P, N - p * P)
        off = p * P + int(rng.integers(0, plen))
        sh[off] ^= 1 << int(rng.integers(0, 8))
    check_checkpoint_parity(cur, sh, P)


def test_no_mutation_empty_log():
    cur = _region(4096 * 300, 1)
    ctx, glog, r, olog, nb = check_checkpoint_parity(cur, cur.clone(), 4096)
    assert r.n_dirty == 0 and r.bytes == 0 and not glog.any()


def test_all_dirty_full_copy_with_tail():
    P, N = 4096, 4096 * 129 + 2048
    cur = _region(N, 2)
    ctx, glog, r, olog, nb = check_checkpoint_parity(cur, ~cur, P)
    n_pages = (N + P - 1) // P
    assert r.n_dirty == n_pages
    g = glog.cpu().numpy()
    payload = np.concatenate([g[i * (16 + P) + 16: i * (16 + P) + 16 + min(P, N - i * P)] for i in range(n_pages)])
    assert np.array_equal(payload, cur.cpu().numpy())


def test_boundary_flips_every_lane_and_bit():
    """byte 0 / P-1, every byte lane of a 16-B vector, every bit; first/last page; adjacent pages."""
    P, n_pages = 4096, 40
    cur = _region(P * n_pages, 3)
    ctx = cc.Context()
    sh = ctx.register_region(1, cur, P)
    log = torch.zeros(n_pages * (16 + P) + 32, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    res = cc.Result()
    cases = []
    for page in (0, 17, n_pages - 1):
        for off in list(range(16)) + [P - 16 + i for i in range(16)] + [2048, 511, 512]:
            cases.append([(page, off, 1 << (off % 8))])
    cases.append([(5, P - 1, 0x80), (6, 0, 0x01)])
    for flips in cases:
        for page, off, mask in flips:
            cur[page * P + off] ^= mask
        ctx.log_reset()
        r = gpu_checkpoint(ctx, 1, 1, res)
        assert ctx.dirty_list(1).tolist() == sorted({f[0] for f in flips})
        assert r.n_dirty == len({f[0] for f in flips})
        assert torch.equal(sh, cur.view(torch.uint8))


def test_bitwise_float_semantics():
    a = torch.zeros(4096, dtype=torch.float32, device="cuda")     # 4 pages of 4 KiB
    ctx = cc.Context()
    ctx.register_region(1, a, 4096)
    ctx.log_attach(torch.zeros(1 << 16, dtype=torch.uint8, device="cuda"))
    a[1500] = -0.0                                                  # +0.0 -> -0.0 is a change
    r = gpu_checkpoint(ctx, 1, 1)
    assert ctx.dirty_list(1).tolist() == [1]
    a.fill_(float("nan"))
    gpu_checkpoint(ctx, 1, 2)
    r = gpu_checkpoint(ctx, 1, 3)                                   # identical NaN payloads are clean
    assert r.n_dirty == 0


def test_log_full_then_retry():
    P = 1024
    cur = _region(P * 64, 4)
    sh = cur.clone()
    for p in (3, 9, 40):
        sh[p * P + 5] ^= 0xFF
    need = 3 * (16 + P) + 32
    ctx = cc.Context()
    shadow = sh.clone()
    ctx.register_region(2, cur, P, shadow=shadow, snapshot_now=False)
    log = torch.zeros(need - 16, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    r = gpu_checkpoint(ctx, 2, 8)
    assert r.status == cc.CC_ERR_LOG_FULL and r.n_dirty == 3 and r.bytes == 0 and r.log_offset_after == 0
    assert not log.any() and torch.equal(shadow, sh)
    log2 = torch.zeros(need, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log2)
    r = gpu_checkpoint(ctx, 2, 8)
    assert r.status == 0 and r.bytes == need
    olog = np.zeros(need, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur.cpu().numpy(), sh.cpu().numpy().copy(), P, 2, 8, olog, 0)
    assert np.array_equal(log2.cpu().numpy(), olog)


def test_consecutive_epochs_chain_offsets_and_two_regions():
    """Several async checkpoints back to back (no host sync between): offsets chain on the device."""
    P1, P2 = 4096, 16384
    a = _region(P1 * 50, 5)
    b = _region(P2 * 20 + 4096, 6)
    ctx = cc.Context()
    sa = ctx.register_region(1, a, P1)
    sb = ctx.register_region(2, b, P2)
    cap = 1 << 20
    log = torch.zeros(cap, dtype=torch.uint8, pin_memory=True)
    ctx.log_attach(log)
    olog = np.zeros(cap, dtype=np.uint8)
    ah, bh = a.cpu().numpy().copy(), b.cpu().numpy().copy()
    sah, sbh = ah.copy(), bh.copy()
    W = 0
    results = [cc.Result() for _ in range(6)]
    expect = []
    for e in range(3):
        a[(7 * e + 3) * P1 + 11] ^= 0x40
        a[49 * P1 + e] ^= 0x01
        b[(e + 20) * P2 + 5 if e == 0 else e * P2 + 100] ^= 0x08
        ah, bh = a.cpu().numpy().copy(), b.cpu().numpy().copy()
        st, D, nb, W = oracle.checkpoint(ah, sah, P1, 1, 10 + e, olog, W)
        expect.append((D.size, nb, W))
        st, D, nb, W = oracle.checkpoint(bh, sbh, P2, 2, 10 + e, olog, W)
        expect.append((D.size, nb, W))
        ctx.checkpoint_delta(1, 10 + e, results[2 * e])
        ctx.checkpoint_delta(2, 10 + e, results[2 * e + 1])
    torch.cuda.synchronize()
    for r, (k, nb, w) in zip(results, expect):
        rr = r.read()
        assert (rr.n_dirty, rr.bytes, rr.log_offset_after, rr.status) == (k, nb, w, 0)
    assert np.array_equal(log.numpy(), olog)


@pytest.mark.parametrize("cfg", ["c1", "c2s", "c3", "c4s"])
def test_scaled_configs(cfg):
    """BASELINE.json configs 1-4: C1 and C3 at full size, C2 and C4 scaled (same structure)."""
    if cfg == "c1":
        P = 4096
        cur = synth.raw_region(64 << 20, 1001, "cuda")
        sh = cur.clone()
        pages = synth.mutate_byte_flips(cur, P, 0.01, 1001)
        assert len(pages) == 164
    elif cfg == "c2s":
        P = 65536
        cur = synth.kv_cache_region(4, 512, 1002, "cuda")
        sh = cur.clone()
        pages = synth.kv_decode_step(cur, 4, 512, 64, 1002)
        assert len(pages) == 256
    elif cfg == "c3":
        P = 65536
        cur = synth.lora_region(32, 1003, "cuda")
        assert cur.numel() == 64 << 20
        sh = cur.clone()
        pages = synth.lora_update(cur, P, 0.05, 1003)
        assert len(pages) == 52
    else:
        P = 16384
        cur = synth.bf16_normal_region(256 << 20, 1004, "cuda")
        sh = cur.clone()
        pages, _, _ = synth.sparse_xor_flips(cur, P, 0.001, 1004)
    cap = len(pages) * (16 + P) + 32
    ctx, glog, r, olog, nb = check_checkpoint_parity(cur, sh, P, log_capacity=cap, pinned_log=(cfg == "c1"))
    assert ctx.dirty_list(3).tolist() == pages.tolist()
    assert nb == cap
    # an immediate second checkpoint is empty
    r2 = gpu_checkpoint(ctx, 3, 18)
    assert r2.n_dirty == 0 and r2.bytes == 0 and r2.log_offset_after == nb


def test_scan_only_leaves_everything_alone():
    P = 4096
    cur = _region(P * 100, 9)
    ctx = cc.Context()
    sh = ctx.register_region(1, cur, P)
    log = torch.zeros(1 << 16, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    cur[5 * P] ^= 1
    cur[77 * P + 9] ^= 1
    sh0 = sh.clone()
    res = cc.Result()
    ctx.scan_only(1, res)
    torch.cuda.synchronize()
    r = res.read()
    assert r.n_dirty == 2 and ctx.dirty_list(1).tolist() == [5, 77]
    assert torch.equal(sh, sh0) and not log.any()
    r = gpu_checkpoint(ctx, 1, 1)
    assert r.n_dirty == 2 and r.bytes == 2 * (16 + P) + 32


def test_argument_errors():
    ctx = cc.Context()
    cur = _region(4096 * 4, 10)
    with pytest.raises(cc.ConcordiaError) as e:
        ctx.checkpoint_delta(9, 1)
    assert e.value.code == cc.CC_ERR_NOT_REGISTERED
    ctx.register_region(1, cur, 4096)
    with pytest.raises(cc.ConcordiaError) as e:
        ctx.register_region(1, cur, 4096)
    assert e.value.code == cc.CC_ERR_EXISTS
    with pytest.raises(cc.ConcordiaError):
        ctx.register_region(2, cur, 100)            # page size not a multiple of 16
    with pytest.raises(cc.ConcordiaError):
        ctx.register_region(0, cur, 4096)           # reserved id
    # checkpoint without a log: k > 0 -> LOG_FULL, nothing happens
    cur[0] ^= 1
    r = gpu_checkpoint(ctx, 1, 1)
    assert r.status == cc.CC_ERR_LOG_FULL and r.n_dirty == 1


def test_log_mirror_drain_by_the_copy_engine():
    """Device log + host mirror: after every epoch the committed bytes are handed to the copy engine; the mirror and its
    published offset follow the oracle's log; reset rewinds both; argument errors."""
    P, n_pages = 4096, 600
    cur = _region(P * n_pages, 21)
    ctx = cc.Context()
    sh = ctx.register_region(1, cur, P)
    cap = 4 << 20
    log = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    mirror = torch.zeros(cap, dtype=torch.uint8, pin_memory=True)
    pub = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(log)
    ctx.log_mirror_attach(mirror, pub)
    copy_stream = torch.cuda.Stream()
    host_cur = cur.cpu().numpy().copy()
    host_sh = host_cur.copy()
    olog = np.zeros(cap, np.uint8)
    rng = np.random.default_rng(4)
    res = cc.Result()
    W = 0
    for e in range(6):
        for p in rng.integers(0, n_pages, 20).tolist():
            off = p * P + int(rng.integers(0, P))
            host_cur[off] ^= 0x33
            cur[off] ^= 0x33
        res.clear()
        ctx.checkpoint_delta(1, e, res)
        torch.cuda.current_stream().synchronize()
        r = res.read()
        st, D, nb, W = oracle.checkpoint(host_cur, host_sh, P, 1, e, olog, W)
        assert (r.status, r.n_dirty, r.log_offset_after) == (st, D.size, W)
        ctx.log_drain(r.log_offset_after, copy_stream)
        if e == 2:
            ctx.log_drain(r.log_offset_after, copy_stream)          # nothing new: a no-op
    copy_stream.synchronize()
    assert int(pub.item()) == W and np.array_equal(mirror.numpy()[:W], olog[:W]) and not mirror[W:].any()
    with pytest.raises(cc.ConcordiaError):
        ctx.log_drain(W - 16, copy_stream)                           # going backwards
    with pytest.raises(cc.ConcordiaError):
        ctx.log_drain(cap + 16, copy_stream)                         # beyond the log
    ctx.log_reset()
    assert int(pub.item()) == 0
    cur[7] ^= 1
    host_cur[7] ^= 1
    res.clear()
    ctx.checkpoint_delta(1, 9, res)
    torch.cuda.current_stream().synchronize()
    r = res.read()
    st, D, nb, W = oracle.checkpoint(host_cur, host_sh, P, 1, 9, olog, 0)
    ctx.log_drain(r.log_offset_after, copy_stream)
    copy_stream.synchronize()
    assert int(pub.item()) == W == 16 + P + 32 and np.array_equal(mirror.numpy()[:W], olog[:W])
    # a mirror smaller than the committed prefix
    small = torch.zeros(W - 16, dtype=torch.uint8, pin_memory=True)
    ctx.log_mirror_attach(small)
    with pytest.raises(cc.ConcordiaError) as ei:
        ctx.log_drain(W, copy_stream)
    assert ei.value.code == cc.CC_ERR_LOG_FULL
    ctx.log_mirror_attach(None)
    with pytest.raises(cc.ConcordiaError):
        ctx.log_drain(W, copy_stream)
    ctx.shutdown()


def test_library_side_drainer_thread_follows_commits_and_resets():
    """cc_log_drain_start: a host thread follows the published committed offset; the host mirror equals the oracle's
    log after every generation, with no per-step drain call -- host-launched checkpoints, then the same through the
    ring / persistent worker, with log resets in between."""
    P, n_pages = 4096, 600
    cur = _region(P * n_pages, 22)
    ctx = cc.Context(ring_capacity=16, max_lifetime_ns=int(60e9))
    ctx.register_region(1, cur, P)
    cap = 4 << 20
    log = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    mirror = torch.zeros(cap, dtype=torch.uint8, pin_memory=True)
    pub = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(log)
    ctx.log_mirror_attach(mirror, pub)
    with pytest.raises(cc.ConcordiaError):
        ctx.log_drain_stop()                                        # not running
    ctx.log_drain_start()
    with pytest.raises(cc.ConcordiaError):
        ctx.log_drain_start()                                       # already running
    with pytest.raises(cc.ConcordiaError):
        ctx.log_drain(16, torch.cuda.Stream())                      # manual drains are refused meanwhile
    host_cur = cur.cpu().numpy().copy()
    host_sh = host_cur.copy()
    rng = np.random.default_rng(5)
    res = cc.Result()

    def mutate():
        for p in rng.integers(0, n_pages, 20).tolist():
            off = p * P + int(rng.integers(0, P))
            host_cur[off] ^= 0x33
            cur[off] ^= 0x33
        torch.cuda.synchronize()

    for generation in range(2):                                     # host-launched, with a reset in between
        olog = np.zeros(cap, np.uint8)
        W = 0
        for e in range(4):
            mutate()
            ctx.checkpoint_delta(1, 10 * generation + e, res)
            st, D, nb, W = oracle.checkpoint(host_cur, host_sh, P, 1, 10 * generation + e, olog, W)
        ctx.log_drain_wait(W, 20.0)
        assert int(pub.item()) == W and np.array_equal(mirror.numpy()[:W], olog[:W])
        (ctx.log_reset if generation == 0 else ctx.log_reset_async)()
    torch.cuda.synchronize()
    # the worker publishes through the same word
    ctx.worker_start()
    try:
        ctx.wait(ctx.submit(cc.CC_TASK_LOG_RESET), 10.0)
        olog = np.zeros(cap, np.uint8)
        W = 0
        for e in range(3):
            A, h = 77, 1000 + e
            ctx.wait(ctx.submit(cc.CC_TASK_TEST_MUTATE, region_id=1, arg0=9, arg1=A, arg2=h), 10.0)
            for j in range(9):
                host_cur[((j * A + h) % n_pages) * P + (h + j) % P] ^= 0x5A
            r = ctx.wait(ctx.submit(cc.CC_TASK_DELTA_CKPT, region_id=1, epoch=50 + e), 10.0)
            st, D, nb, W = oracle.checkpoint(host_cur, host_sh, P, 1, 50 + e, olog, W)
            assert (r.status, r.n_dirty, r.log_offset_after) == (st, D.size, W)
        ctx.log_drain_wait(W, 20.0)
        assert int(pub.item()) == W and np.array_equal(mirror.numpy()[:W], olog[:W])
    finally:
        ctx.worker_stop()
    ctx.log_drain_stop()
    ctx.shutdown()


@pytest.mark.parametrize("path", ["phases", "single", "small"])
def test_host_sees_every_record_byte_once_the_committed_offset_moves(path):
    """PAPER.md:L263 "a commit marker publishes the epoch only after all bytes are visible": records go straight into a
    PINNED HOST log; the host never synchronises with the stream -- it polls the committed-offset word and, the moment it
    moves, replays the newly committed bytes with the oracle's applier (every record's CRC32C is checked there) onto its own
    copy of the region.  The record bytes are written by hundreds of blocks; only the last one executes a system-scope fence
    (the others release at gpu scope), so this is the test of that fence chain."""
    P, n_pages, per_step, steps = 4096, 4096, 384, 40
    N = P * n_pages
    cur = _region(N, 77)
    host = cur.cpu().numpy().copy()                     # what the host has recovered so far
    ctx = cc.Context()
    ctx.register_region(1, cur, P)
    cap = steps * (per_step * (16 + P) + 32) + 4096
    hlog = torch.zeros(cap, dtype=torch.uint8, pin_memory=True)
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(hlog, committed)
    log_np, com_np = hlog.numpy(), committed.numpy()
    kw = {"phases": cc.CC_PATH_PHASES, "single": cc.CC_PATH_SINGLE_PASS, "small": cc.CC_PATH_SMALL}[path]
    rng = np.random.default_rng(9)
    import time
    W = 0
    for it in range(steps):
        pages = torch.from_numpy(rng.choice(n_pages, per_step, replace=False)).cuda()
        offs = pages * P + torch.from_numpy(rng.integers(0, P, per_step)).cuda()
        cur[offs] ^= 0x5A
        ctx.checkpoint_ex(1, it, None, path=kw)         # no result, no synchronize
        need = per_step * (16 + P) + 32
        t0 = time.time()
        while int(com_np[0]) < W + need:
            assert time.time() - t0 < 20, "committed offset never moved"
        st, nrec, consumed = oracle.apply_log(log_np[W:W + need], need, [oracle.Region(1, P, host)])
        assert (st, nrec, consumed) == (0, per_step, need), (it, st, nrec, consumed)
        W += need
    torch.cuda.synchronize()
    assert np.array_equal(host, cur.cpu().numpy())
