"""GPU parity for run-length records: the applier and the compactor on run logs
written by the ORACLE, and cc_checkpoint_delta_rle against oracle.checkpoint_rle, bit-exact."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc

pytestmark = pytest.mark.gpu


def _history(P, n_pages, tail, R, seed, epochs=3):
    """A few epochs of clustered changes written by the oracle with run records.  Returns (old, final, log, W, n_records)."""
    N = (n_pages - 1) * P + (tail or P)
    rng = np.random.default_rng(seed)
    old = rng.integers(0, 256, N, dtype=np.uint8)
    cur, sh = old.copy(), old.copy()
    log = np.zeros(epochs * (N + 16 * n_pages + 64), np.uint8)
    W, n_rec = 0, 0
    for e in range(epochs):
        for _ in range(max(1, n_pages // 12)):
            a = int(rng.integers(0, n_pages))
            for p in range(a, min(n_pages, a + int(rng.integers(1, 7)))):      # clusters -> runs
                cur[p * P + int(rng.integers(0, min(P, N - p * P)))] ^= 0x81
        cur[N - 1] ^= 1                                                         # the tail page every epoch (duplicates)
        st, D, runs, nb, W = oracle.checkpoint_rle(cur, sh, P, 4, 10 + e, R, log, W)
        assert st == 0
        n_rec += runs
    return old, cur, log, W, n_rec


@pytest.mark.parametrize("P,n_pages,tail,R", [(16, 40, 0, 4), (64, 300, 48, 8), (4096, 400, 1024, 16), (4112, 60, 16, 4),
                                              (16384, 100, 4096 + 16, 64), (65536, 48, 65520, 16), (81920, 20, 4096, 2)])
@pytest.mark.parametrize("pinned", [False, True])
def test_apply_and_compact_run_logs_written_by_the_oracle(P, n_pages, tail, R, pinned):
    old, final, olog, W, n_rec = _history(P, n_pages, tail, R, P + n_pages)
    N = old.size
    work = torch.from_numpy(old.copy()).cuda()
    ctx = cc.Context()
    sh = ctx.register_region(4, work, P)
    ctx.apply_attach(n_rec + 16)
    lt = torch.from_numpy(olog[:W].copy())
    lt = lt.pin_memory() if pinned else lt.cuda()
    res = cc.Result()
    # compaction first (must not touch the region), against the oracle's
    exp = np.zeros(N + 16 * n_pages + 64, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(olog, W, [oracle.Region(4, P, np.zeros(N, np.uint8))], exp)
    out = torch.zeros(exp.size, dtype=torch.uint8, device="cuda")
    ctx.compact_log(lt, W, out, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (st, n_out, nb, consumed) == (0, n_out, nb, W), r.as_dict()
    assert np.array_equal(out.cpu().numpy(), exp) and np.array_equal(work.cpu().numpy(), old)
    # replay of the run log
    host = old.copy()
    e = oracle.apply_log(olog, W, [oracle.Region(4, P, host)])
    res.clear()
    ctx.apply_log(lt, W, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes) == e == (0, n_rec, W), r.as_dict()
    assert np.array_equal(work.cpu().numpy(), host) and np.array_equal(host, final) and torch.equal(sh, work)
    # truncated inside the last run record: that epoch is not applied
    work.copy_(torch.from_numpy(old))
    host = old.copy()
    cut = W - 32 - 24
    e = oracle.apply_log(olog, cut, [oracle.Region(4, P, host)])
    res.clear()
    ctx.apply_log(lt, cut, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes) == e and np.array_equal(work.cpu().numpy(), host)
    # a flipped bit in the middle of a run payload: CORRUPT, same prefix as the oracle
    bad = olog[:W].copy()
    bad[W // 2] ^= 0x10
    work.copy_(torch.from_numpy(old))
    host = old.copy()
    e = oracle.apply_log(bad, W, [oracle.Region(4, P, host)])
    bt = torch.from_numpy(bad).cuda()
    res.clear()
    ctx.apply_log(bt, W, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes) == e and np.array_equal(work.cpu().numpy(), host)
    ctx.shutdown()


def test_malformed_run_lengths_are_corrupt():
    import struct
    P, n_pages = 4096, 8
    N = P * n_pages - 2048
    cur = synth.raw_region(N, 5, "cuda")
    ctx = cc.Context()
    ctx.register_region(4, cur, P)
    ctx.apply_attach(64)
    res = cc.Result()
    before = cur.clone()
    for page, length, ok in ((2, 3 * P, True), (6, P + P - 2048, True), (2, P + 16, False), (6, 2 * P, False), (8, P, False), (3, 0, False)):
        payload = np.full(length, 7, np.uint8)
        rec = struct.pack("<IIII", 4, page, length, oracle.crc32c(payload)) + payload.tobytes()
        cp = struct.pack("<QII", 1, 4, 1)
        log = np.frombuffer(rec + struct.pack("<IIII", 0xFFFFFFFF, 0xFFFFFFFF, 16, oracle.crc32c(np.frombuffer(cp, np.uint8))) + cp, np.uint8)
        host = before.cpu().numpy().copy()
        e = oracle.apply_log(log, log.size, [oracle.Region(4, P, host)])
        assert (e[0] == 0) == ok
        cur.copy_(before)
        res.clear()
        ctx.apply_log(torch.from_numpy(log.copy()).cuda(), log.size, res)
        torch.cuda.synchronize()
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes) == e, (page, length, r.as_dict(), e)
        assert np.array_equal(cur.cpu().numpy(), host)
    ctx.shutdown()


# ------------------------------------------------------------------ the run-record writer --

def _clustered(P, n_pages, tail, seed, density=10):
    N = (n_pages - 1) * P + (tail or P)
    cur = synth.raw_region(N, seed, "cuda")
    sh = cur.clone()
    rng = np.random.default_rng(seed)
    for _ in range(max(1, n_pages // density)):
        a = int(rng.integers(0, n_pages))
        for p in range(a, min(n_pages, a + int(rng.integers(1, 9)))):
            sh[p * P + int(rng.integers(0, min(P, N - p * P)))] ^= 1 << int(rng.integers(0, 8))
    sh[N - 1] ^= 1
    sh[0] ^= 1
    return cur, sh, N


def _rle_parity(cur, sh0, P, R, cap=None, pinned=False, region_id=4, epoch=31):
    N = cur.numel()
    n_pages = (N + P - 1) // P
    cap = cap if cap is not None else N + 16 * n_pages + 96
    cur_h = cur.cpu().numpy()
    sh_h = sh0.cpu().numpy().copy()
    olog = np.zeros(cap, np.uint8)
    st, D, runs, nb, W = oracle.checkpoint_rle(cur_h, sh_h, P, region_id, epoch, R, olog, 0)
    ctx = cc.Context()
    shadow = sh0.clone()
    ctx.register_region(region_id, cur, P, shadow=shadow, snapshot_now=False)
    glog = torch.zeros(cap, dtype=torch.uint8, pin_memory=True) if pinned else torch.zeros(cap, dtype=torch.uint8, device="cuda")
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(glog, committed)
    res = cc.Result()
    ctx.checkpoint_delta_rle(region_id, epoch, R, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.seq_done, r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch) == (1, st, D.size, nb, W, epoch), r.as_dict()
    assert ctx.dirty_list(region_id).tolist() == D.tolist()
    g = glog.cpu().numpy()
    assert np.array_equal(g, olog), "log bytes differ at %s" % np.nonzero(g != olog)[0][:8]
    assert np.array_equal(shadow.cpu().numpy(), sh_h) and int(committed.item()) == W
    return ctx, r, runs, glog, nb


@pytest.mark.parametrize("P,n_pages,tail,R", [(16, 70, 0, 4), (64, 300, 48, 8), (256, 1100, 0, 32), (4096, 700, 1024, 16),
                                              (4096, 2100, 0, 256), (4112, 60, 16, 4), (16384, 130, 4096 + 16, 64),
                                              (65536, 48, 65520, 16), (65536, 40, 0, 3), (81920, 20, 4096, 2), (1 << 20, 5, 0, 2)])
def test_rle_writer_shapes(P, n_pages, tail, R):
    cur, sh, N = _clustered(P, n_pages, tail, P % 89 + n_pages)
    ctx, r, runs, glog, nb = _rle_parity(cur, sh, P, R, pinned=(n_pages % 2 == 0))
    assert 0 < runs <= r.n_dirty
    # an immediate second call is empty
    res = cc.Result()
    ctx.checkpoint_delta_rle(4, 32, R, res)
    torch.cuda.synchronize()
    r2 = res.read()
    assert (r2.status, r2.n_dirty, r2.bytes, r2.log_offset_after) == (0, 0, 0, nb)
    ctx.shutdown()


def test_rle_run_pages_1_equals_checkpoint_delta_all_dirty_log_full_and_errors():
    P, n_pages = 4096, 515
    N = P * n_pages - 2048
    cur, sh, _ = _clustered(P, n_pages, P - 2048, 9)
    ctx, r, runs, glog, nb = _rle_parity(cur, sh, P, 1)
    assert runs == r.n_dirty
    olog = np.zeros(glog.numel(), np.uint8)
    st, D, nb1, W1 = oracle.checkpoint(cur.cpu().numpy(), sh.cpu().numpy().copy(), P, 4, 31, olog, 0)
    assert nb1 == nb and np.array_equal(glog.cpu().numpy(), olog)
    ctx.shutdown()
    # all dirty: ceil(n_pages / R) records
    ctx, r, runs, glog, nb = _rle_parity(cur, ~cur, P, 64)
    assert r.n_dirty == n_pages and runs == (n_pages + 63) // 64 and nb == N + 16 * runs + 32
    ctx.shutdown()
    # one byte short: LOG_FULL, nothing written
    exact = np.zeros(N + 16 * n_pages + 96, np.uint8)
    st, D, runs, need, W = oracle.checkpoint_rle(cur.cpu().numpy(), sh.cpu().numpy().copy(), P, 4, 31, 16, exact, 0)
    ctx, r, runs, glog, nb = _rle_parity(cur, sh, P, 16, cap=need - 1)
    assert r.status == cc.CC_ERR_LOG_FULL and not glog.any()
    with pytest.raises(cc.ConcordiaError):
        ctx.checkpoint_delta_rle(4, 1, 0)
    with pytest.raises(cc.ConcordiaError):
        ctx.checkpoint_delta_rle(4, 1, (1 << 32) // P + 1)
    ctx.shutdown()


def test_rle_chains_with_other_paths_replays_and_runs_in_the_worker():
    P, n_pages, R = 16384, 256, 8
    cur = synth.raw_region(P * n_pages, 13, "cuda")
    ctx = cc.Context(ring_capacity=8, max_lifetime_ns=int(60e9))
    sh = ctx.register_region(1, cur, P)
    cap = 3 * P * n_pages
    log = torch.zeros(cap, dtype=torch.uint8, pin_memory=True)
    ctx.log_attach(log)
    ctx.apply_attach(4096)
    old = cur.clone()
    host_cur = cur.cpu().numpy().copy()
    host_sh = host_cur.copy()
    olog = np.zeros(cap, np.uint8)
    rng = np.random.default_rng(2)
    W = 0
    res = cc.Result()

    def mutate():
        a = int(rng.integers(0, n_pages - 12))
        for p in range(a, a + int(rng.integers(2, 12))):
            off = p * P + int(rng.integers(0, P))
            host_cur[off] ^= 0x55
            cur[off] ^= 0x55

    for e in range(4):                       # host-launched: rle, plain, rle, fused
        mutate()
        res.clear()
        if e % 2 == 0:
            ctx.checkpoint_delta_rle(1, e, R, res)
            st, D, runs, nb, W = oracle.checkpoint_rle(host_cur, host_sh, P, 1, e, R, olog, W)
        else:
            (ctx.checkpoint_delta if e == 1 else ctx.checkpoint_delta_fused)(1, e, res)
            st, D, nb, W = oracle.checkpoint(host_cur, host_sh, P, 1, e, olog, W)
        torch.cuda.synchronize()
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (st, D.size, nb, W), (e, r.as_dict())
    for e in range(4, 7):                    # through the worker
        mutate()
    torch.cuda.synchronize()
    ctx.worker_start()
    try:
        s = ctx.submit(cc.CC_TASK_DELTA_CKPT, region_id=1, epoch=4, arg0=R, flags=cc.CC_TASKF_RLE)
        r = ctx.wait(s, 20.0)
    finally:
        ctx.worker_stop()
    st, D, runs, nb, W = oracle.checkpoint_rle(host_cur, host_sh, P, 1, 4, R, olog, W)
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (st, D.size, nb, W), r.as_dict()
    assert np.array_equal(log.numpy(), olog) and np.array_equal(sh.cpu().numpy(), host_sh)
    # the mixed log replays onto the old state
    final = cur.clone()
    cur.copy_(old)
    res.clear()
    ctx.apply_log(log, W, res)
    torch.cuda.synchronize()
    assert res.read().status == 0 and torch.equal(cur, final)
    ctx.shutdown()


def test_rle_prefill_shaped_c2_full_size():
    """A prefill-like boundary on the config-2 KV region: 64 sequences each fill 32 CONSECUTIVE blocks of every layer
    (contiguous dirty ranges) -> run records; sampled records against the oracle's CRC."""
    free, _ = torch.cuda.mem_get_info()
    if free < 24 * 2**30:
        pytest.skip("needs 24 GiB of device memory")
    layers, blocks, P, R = 32, 4096, 65536, 16
    cur = synth.kv_cache_region(layers, blocks, 1002, "cuda")
    ctx = cc.Context()
    sh = ctx.register_region(1, cur, P)
    v = cur.view(layers, blocks, P)
    g = synth.gen(77, "cuda")
    starts = (torch.randperm(blocks // 32, generator=g, device="cuda")[:64] * 32 + 5).clamp(max=blocks - 32)
    for s0 in starts.tolist():
        v[:, s0:s0 + 32, :256] = torch.randint(0, 256, (layers, 32, 256), dtype=torch.uint8, device="cuda", generator=g)
    k = layers * 64 * 32
    cap = k * P + 16 * k + 64
    log = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    res = cc.Result()
    ctx.checkpoint_delta_rle(1, 3, R, res)
    torch.cuda.synchronize()
    r = res.read()
    D = ctx.dirty_list(1)
    assert r.status == 0 and r.n_dirty == k == D.numel()
    # expected runs from the generator's own page set: consecutive pages, split at multiples of R
    pages = sorted(l * blocks + b for l in range(layers) for s0 in starts.tolist() for b in range(s0, s0 + 32))
    assert D.tolist() == pages
    n_runs = sum(1 for i, p in enumerate(pages) if i == 0 or pages[i - 1] + 1 != p or p % R == 0)
    assert n_runs < k // 8 and r.bytes == k * P + 16 * n_runs + 32
    assert torch.equal(sh, cur)
    # walk the first records and check header + CRC against the oracle
    off = 0
    for _ in range(6):
        hdr = log[off:off + 16].cpu().numpy().view(np.uint32)
        rid, p0, ln, crc = [int(x) for x in hdr]
        assert rid == 1 and ln % P == 0 and ln // P in (5, 11, 16)
        payload = log[off + 16:off + 16 + ln].cpu().numpy()
        assert crc == oracle.crc32c(payload) and np.array_equal(payload, cur[p0 * P:p0 * P + ln].cpu().numpy())
        off += 16 + ln
    ctx.shutdown()


@pytest.mark.parametrize("R", [3, 5, 7])
def test_rle_millions_of_small_pages_with_odd_run_lengths(R):
    """More than 2^22 pages with a run length that is no power of two: the single pass must still cut the region into at
    most 2^20 warp tiles (its look-back table), i.e. round the tile size UP to a multiple of R, not down."""
    P, n_pages = 16, (1 << 22) + 37
    N = n_pages * P
    cur = synth.raw_region(N, 77 + R, "cuda")
    sh = cur.clone()
    rng = np.random.default_rng(R)
    starts = rng.choice(n_pages - 16, 3000, replace=False)
    pages = np.unique(np.concatenate([starts + j for j in range(int(R) + 2)] + [np.array([0, n_pages - 1, n_pages - 2])]))
    idx = torch.from_numpy(pages * P + rng.integers(0, P, pages.size)).cuda()
    sh[idx] = sh[idx] ^ 0x40
    ctx, r, runs, glog, nb = _rle_parity(cur, sh, P, R, cap=pages.size * (16 + P) + 4096)
    assert r.n_dirty == pages.size and 0 < runs < pages.size
    ctx.shutdown()
