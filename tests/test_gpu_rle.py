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
