"""GPU parity: cc_apply_log vs the CPU apply oracle (post-apply region, shadow, counters, status)."""
import struct

import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc
from gpu_util import gpu_checkpoint

pytestmark = pytest.mark.gpu


def _gpu_apply(ctx, log_t, nbytes):
    res = cc.Result()
    ctx.apply_log(log_t, nbytes, res)
    torch.cuda.synchronize()
    r = res.read()
    assert r.seq_done == 1
    return r


def _two_epoch_setup(P=64, n_pages=12, tail=32):
    N = (n_pages - 1) * P + tail
    rng = np.random.default_rng(5)
    old = rng.integers(0, 256, N, dtype=np.uint8)
    cur, sh = old.copy(), old.copy()
    log = np.zeros(4096, dtype=np.uint8)
    for p in (1, 4, n_pages - 1):
        cur[p * P + 3] ^= 0x55
    st, D1, nb1, W = oracle.checkpoint(cur, sh, P, 3, 100, log, 0)
    for p in (4, 7):
        cur[p * P + 9] ^= 0xAA
    st, D2, nb2, W = oracle.checkpoint(cur, sh, P, 3, 101, log, W)
    return old, log, nb1, nb2, P


def _compare(old, log_np, nbytes, P, region_id=3, pinned=False, max_records=1024):
    """Apply log_np[:nbytes] to `old` on both sides and compare everything."""
    reg_o, sh_o = old.copy(), old.copy()
    exp = oracle.apply_log(log_np, nbytes, [oracle.Region(region_id, P, reg_o, sh_o)])
    ctx = cc.Context()
    reg = torch.from_numpy(old.copy()).cuda()
    sh = ctx.register_region(region_id, reg, P)
    ctx.apply_attach(max_records)
    lt = torch.from_numpy(log_np.copy())
    lt = lt.pin_memory() if pinned else lt.cuda()
    r = _gpu_apply(ctx, lt, nbytes)
    assert (r.status, r.n_dirty, r.bytes) == exp, ((r.status, r.n_dirty, r.bytes), exp)
    assert np.array_equal(reg.cpu().numpy(), reg_o)
    assert np.array_equal(sh.cpu().numpy(), sh_o)
    return ctx, reg, sh, r


def test_round_trip_idempotent_then_empty_checkpoint():
    old, log, nb1, nb2, P = _two_epoch_setup()
    ctx, reg, sh, r = _compare(old, log, nb1 + nb2, P)
    assert r.epoch == 2
    lt = torch.from_numpy(log).cuda()
    before = reg.clone()
    r = _gpu_apply(ctx, lt, nb1 + nb2)                      # idempotent
    assert torch.equal(reg, before) and r.n_dirty == 5
    ctx.log_attach(torch.zeros(4096, dtype=torch.uint8, device="cuda"))
    r = gpu_checkpoint(ctx, 3, 200)                          # apply refreshed the shadow
    assert r.n_dirty == 0 and r.bytes == 0


def test_truncation_sweep():
    old, log, nb1, nb2, P = _two_epoch_setup()
    total = nb1 + nb2
    ctx = cc.Context()
    reg = torch.from_numpy(old.copy()).cuda()
    sh = ctx.register_region(3, reg, P)
    ctx.apply_attach(64)
    lt = torch.from_numpy(log).cuda()
    old_t = torch.from_numpy(old).cuda()
    for t in list(range(0, total + 1, 7)) + [nb1 - 1, nb1, nb1 + 1, total - 1, total]:
        reg.copy_(old_t)
        sh.copy_(old_t)
        reg_o = old.copy()
        exp = oracle.apply_log(log, t, [oracle.Region(3, P, reg_o)])
        r = _gpu_apply(ctx, lt, t)
        assert (r.status, r.n_dirty, r.bytes) == exp, t
        assert np.array_equal(reg.cpu().numpy(), reg_o), t


@pytest.mark.parametrize("where,idx,val", [("payload1", None, None), ("payload2", None, None),
                                           ("hdr2", 0, 99), ("hdr2", 4, 10_000), ("hdr2", 8, 48),
                                           ("hdr2", 12, 0xDEADBEEF), ("hdr2", 8, 1 << 30),
                                           ("commit_k", None, None), ("commit_region", None, None),
                                           ("commit_crc", None, None), ("commit_pageidx", None, None),
                                           ("commit_len", None, None)])
def test_corruption_cases(where, idx, val):
    old, log, nb1, nb2, P = _two_epoch_setup()
    bad = log.copy()
    c = nb1 + nb2 - 32
    if where == "payload1":
        bad[16] ^= 0x80
    elif where == "payload2":
        bad[nb1 + 16 + 5] ^= 0x04
    elif where == "hdr2":
        bad[nb1 + idx: nb1 + idx + 4] = np.frombuffer(struct.pack("<I", val), dtype=np.uint8)
    elif where in ("commit_k", "commit_region"):
        payload = struct.pack("<QII", 101, 3, 3) if where == "commit_k" else struct.pack("<QII", 101, 4, 2)
        bad[c + 16: c + 32] = np.frombuffer(payload, dtype=np.uint8)
        bad[c + 12: c + 16] = np.frombuffer(struct.pack("<I", oracle.crc32c(payload)), dtype=np.uint8)
    elif where == "commit_crc":
        bad[c + 20] ^= 1
    elif where == "commit_pageidx":
        bad[c + 4] = 0
    else:
        bad[c + 8] = 32
    _compare(old, bad, nb1 + nb2, P)


def test_config5a_scaled_mixed_pages_duplicates(pinned=False):
    """Config 5a scaled: three regions (4/16/64 KiB pages) of one arena, log written by the ORACLE's record
    writer, pages repeat across epochs (last wins).  Log in device memory and in pinned host memory."""
    arena_bytes = 64 << 20
    arena = synth.raw_region(arena_bytes, 1005, "cuda")
    unit = arena_bytes // 8
    eps = synth.recovery_epochs(arena_bytes, 30, 40, 1005, forced_repeats=10)
    cap = sum(e.payloads.numel() + 16 * e.pages.numel() + 32 for e in eps)
    olog = np.zeros(cap, dtype=np.uint8)
    W = 0
    views = {rid: (o8 * unit, s8 * unit, P) for rid, o8, s8, P in synth.C5A_REGIONS}
    for e in eps:
        o, sz, P = views[e.region_id]
        st, W = oracle.write_epoch(olog, W, e.region_id, e.epoch, sz, P, e.pages.numpy(), e.payloads.numpy())
        assert st == 0
    assert W == cap
    host = arena.cpu().numpy().copy()
    regs_o = [oracle.Region(rid, P, host[o:o + sz]) for rid, (o, sz, P) in views.items()]
    exp = oracle.apply_log(olog, W, regs_o)
    assert exp[0] == 0 and exp[1] == sum(e.pages.numel() for e in eps)

    for pinned, staged in ((False, False), (True, False), (True, True), (False, True)):
        work = arena.clone()
        ctx = cc.Context()
        shadows = {}
        for rid, (o, sz, P) in views.items():
            shadows[rid] = ctx.register_region(rid, work[o:o + sz], P)
        ctx.apply_attach(exp[1] + 64)
        if staged:
            ctx.apply_stage_attach(W)          # host logs cross the link once (copy engine); device logs are unaffected
        lt = torch.from_numpy(olog)
        lt = lt.pin_memory() if pinned else lt.cuda()
        r = _gpu_apply(ctx, lt, W)
        assert (r.status, r.n_dirty, r.bytes, r.epoch) == (0, exp[1], W, len(eps))
        assert np.array_equal(work.cpu().numpy(), host)
        for rid, (o, sz, P) in views.items():
            assert np.array_equal(shadows[rid].cpu().numpy(), host[o:o + sz])
        # the staging buffer's use is visible: only a host-resident log with a buffer attached counts
        assert ctx.apply_stage_stats() == ((1, 0) if pinned and staged else (0, 0))
        if pinned and staged:
            ctx.apply_stage_attach(W - 16)     # one unit too small: the log is read in place -- correct, and counted
            work.copy_(arena)
            r = _gpu_apply(ctx, lt, W)
            assert (r.status, r.n_dirty, r.bytes) == (0, exp[1], W) and np.array_equal(work.cpu().numpy(), host)
            assert ctx.apply_stage_stats() == (1, 1)
        ctx.shutdown()


def test_scratch_too_small_applies_nothing():
    P, n_pages = 64, 600
    cur = synth.raw_region(P * n_pages, 78, "cuda")
    old = (~cur).contiguous()
    olog = np.zeros(n_pages * (16 + P) + 32, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur.cpu().numpy(), old.cpu().numpy().copy(), P, 3, 1, olog, 0)
    ctx = cc.Context()
    reg = old.clone()
    ctx.register_region(3, reg, P)
    ctx.apply_attach(100)                       # room for ~100 records, the log holds 600
    r = _gpu_apply(ctx, torch.from_numpy(olog).cuda(), nb)
    assert r.status == cc.CC_ERR_SCRATCH and r.n_dirty == 0 and r.bytes == 0
    assert torch.equal(reg, old)


def test_checkpoint_then_apply_round_trip_c1():
    """Config 1 round trip: GPU checkpoint log applied by the GPU applier onto the old snapshot."""
    P = 4096
    cur = synth.raw_region(64 << 20, 1001, "cuda")
    old = cur.clone()
    pages = synth.mutate_byte_flips(cur, P, 0.01, 1001)
    ctx = cc.Context()
    ctx.register_region(1, cur, P, shadow=old.clone(), snapshot_now=False)
    log = torch.zeros(len(pages) * (16 + P) + 32, dtype=torch.uint8, pin_memory=True)
    ctx.log_attach(log)
    r = gpu_checkpoint(ctx, 1, 1)
    assert r.n_dirty == len(pages) and r.bytes == log.numel()
    ctx2 = cc.Context()
    target = old.clone()
    ctx2.register_region(1, target, P)
    ctx2.apply_attach(1000)
    r2 = _gpu_apply(ctx2, log, log.numel())
    assert (r2.status, r2.n_dirty, r2.bytes) == (0, len(pages), log.numel())
    assert torch.equal(target, cur)
    # and the oracle agrees about the same log
    host = old.cpu().numpy().copy()
    assert oracle.apply_log(log.numpy(), log.numel(), [oracle.Region(1, P, host)]) == (0, len(pages), log.numel())
    assert np.array_equal(host, cur.cpu().numpy())


def test_long_single_epoch_many_parse_steps():
    """More records in one epoch than the parser's speculation width, with a short tail page last."""
    P, n_pages = 64, 3000
    N = (n_pages - 1) * P + 32
    cur = synth.raw_region(N, 77, "cuda")
    old = (~cur).contiguous()
    olog = np.zeros(n_pages * (16 + P) + 32, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur.cpu().numpy(), old.cpu().numpy().copy(), P, 3, 1, olog, 0)
    assert D.size == n_pages
    ctx = cc.Context()
    reg = old.clone()
    ctx.register_region(3, reg, P)
    ctx.apply_attach(4000)
    r = _gpu_apply(ctx, torch.from_numpy(olog).cuda(), nb)
    assert (r.status, r.n_dirty, r.bytes) == (0, n_pages, nb)
    assert torch.equal(reg, cur)


@pytest.mark.parametrize("bad_epoch", [0, 1, 2, 3, 4])
def test_failed_check_falls_back_to_the_latest_committed_record(bad_epoch):
    """Five epochs rewrite overlapping pages; one payload bit of epoch `bad_epoch` is flipped.  Pages whose LATEST record
    lies in or behind the damaged epoch must end up with their latest COMMITTED record (or untouched) -- the case in which
    the applier's side-by-side validation + scatter has to rebuild its last-wins table over the committed prefix.  The same
    context then applies the undamaged log (the tables must have been left clean)."""
    P, n_pages = 4096, 64
    N = P * n_pages
    rng = np.random.default_rng(17)
    old = rng.integers(0, 256, N, dtype=np.uint8)
    cur, sh = old.copy(), old.copy()
    log = np.zeros(1 << 20, dtype=np.uint8)
    W, ends = 0, []
    for e in range(5):
        for p in sorted(set(rng.integers(0, n_pages, 12).tolist()) | {5, 6 + e}):     # page 5 in every epoch
            cur[p * P + int(rng.integers(0, P))] ^= 0x3C
        st, D, nb, W = oracle.checkpoint(cur, sh, P, 3, 200 + e, log, W)
        assert st == 0
        ends.append(W)
    good = log.copy()
    start = ends[bad_epoch - 1] if bad_epoch else 0
    log[start + 16 + 100] ^= 0x04                      # first record's payload of the damaged epoch
    ctx, reg, sh_t, r = _compare(old, log, W, P)
    assert r.status == cc.CC_ERR_CORRUPT and r.epoch == bad_epoch
    # the same context, the undamaged log, from scratch
    reg.copy_(torch.from_numpy(old).cuda())
    sh_t.copy_(torch.from_numpy(old).cuda())
    r2 = _gpu_apply(ctx, torch.from_numpy(good).cuda(), W)
    reg_o, sh_o = old.copy(), old.copy()
    exp = oracle.apply_log(good, W, [oracle.Region(3, P, reg_o, sh_o)])
    assert (r2.status, r2.n_dirty, r2.bytes) == exp and r2.status == 0 and r2.epoch == 5
    assert np.array_equal(reg.cpu().numpy(), reg_o) and np.array_equal(sh_t.cpu().numpy(), sh_o)
    assert np.array_equal(reg_o, cur)


def _commit_image(epoch, region_id, k):
    """the 32 bytes of a VALID commit record (signature, length 16, CRC32C of its payload)"""
    pay = struct.pack("<QII", epoch, region_id, k)
    return struct.pack("<IIII", 0xFFFFFFFF, 0xFFFFFFFF, 16, oracle.crc32c(np.frombuffer(pay, np.uint8))) + pay


@pytest.mark.parametrize("n_false,max_records", [(1, 1024), (7, 1024), (300, 64)])
def test_payloads_that_contain_valid_commit_record_images(n_false, max_records):
    """The parallel parse finds commit records by signature + CRC; a page whose BYTES contain a valid commit record puts a
    false candidate on its list.  The epoch walks must notice (they run past the false one) and hand the log to the serial
    parser: same result as the sequential definition.  (300 false candidates with tables for 64 records: the candidate list
    overflows, which must end the same way.)"""
    P, n_pages = 4096, 48
    N = P * n_pages
    rng = np.random.default_rng(n_false)
    old = rng.integers(0, 256, N, dtype=np.uint8)
    cur, sh = old.copy(), old.copy()
    log = np.zeros(1 << 20, dtype=np.uint8)
    W, placed = 0, 0
    for e in range(6):
        pages = sorted(set(rng.integers(0, n_pages, 5).tolist()))
        for p in pages:
            cur[p * P + int(rng.integers(0, P))] ^= 0x42
            per_page = min(n_false - placed, 60) if e % 2 == 0 else 0
            for q in range(per_page):                     # images at 16-byte-aligned offsets of the page
                off = p * P + 64 * q + 16 * (q % 2)
                img = np.frombuffer(_commit_image(int(rng.integers(0, 1 << 40)), int(rng.integers(1, 9)), int(rng.integers(0, 9))), np.uint8)
                cur[off:off + 32] = img
            placed += per_page
        st, D, nb, W = oracle.checkpoint(cur, sh, P, 3, 300 + e, log, W)
        assert st == 0
    assert placed == n_false
    ctx, reg, sh_t, r = _compare(old, log, W, P, max_records=max_records)
    assert r.status == 0 and r.epoch == 6
    # a torn tail behind the false candidates, and a damaged real commit record
    _compare(old, log, W - 40, P, max_records=max_records)
    bad = log.copy()
    bad[W - 4] ^= 0x80                                     # k of the last commit record
    _compare(old, bad, W, P, max_records=max_records)


def test_thousands_of_one_record_epochs():
    """3,000 epochs of one or two 64-byte-page records: 3,000 candidates ranked over several tiles, 3,000 epoch walks
    chained by look-back."""
    P, n_pages, E = 64, 512, 3000
    N = P * n_pages
    rng = np.random.default_rng(12)
    old = rng.integers(0, 256, N, dtype=np.uint8)
    cur, sh = old.copy(), old.copy()
    log = np.zeros(E * (2 * (16 + P) + 32) + 64, dtype=np.uint8)
    W = 0
    for e in range(E):
        for p in rng.integers(0, n_pages, 1 + e % 2).tolist():
            cur[p * P + int(rng.integers(0, P))] ^= 0x01
        st, D, nb, W = oracle.checkpoint(cur, sh, P, 3, e, log, W)
    ctx, reg, sh_t, r = _compare(old, log, W, P, max_records=8192)
    assert r.status == 0 and r.epoch >= E - 600 and np.array_equal(reg.cpu().numpy(), cur)
    _compare(old, log, W // 2 + 8, P, max_records=8192)    # torn in the middle


def test_more_epochs_than_the_candidate_ranking_takes_go_to_the_serial_parser():
    """140,000 one-record epochs of 16-byte pages: more commit records than the quadratic ranking of the parallel parse
    accepts (2^17), so the whole log is parsed by the linear serial parser -- same result as the oracle, and the same
    context then takes a short log through the parallel parse again (the overflow flag was re-armed)."""
    P, n_pages, E = 16, 64, 140_000
    N = P * n_pages
    rng = np.random.default_rng(140)
    old = rng.integers(0, 256, N, dtype=np.uint8)
    cur, sh = old.copy(), old.copy()
    log = np.zeros(E * (16 + P + 32) + 64, dtype=np.uint8)
    W = 0
    where = rng.integers(0, N, E)
    for e in range(E):
        cur[where[e]] ^= 0x01 + (e & 0x7E)
        st, D, nb, W = oracle.checkpoint(cur, sh, P, 3, e, log, W)
        assert D.size == 1
    ctx, reg, sh_t, r = _compare(old, log, W, P, max_records=E + 64)
    assert (r.status, r.n_dirty, r.epoch, r.bytes) == (0, E, E, W) and np.array_equal(reg.cpu().numpy(), cur)
    short = 50 * (16 + P + 32)
    reg_o, sh_o = old.copy(), old.copy()
    exp = oracle.apply_log(log, short, [oracle.Region(3, P, reg_o, sh_o)])
    reg.copy_(torch.from_numpy(old))
    sh_t.copy_(torch.from_numpy(old))
    r = _gpu_apply(ctx, torch.from_numpy(log[:short].copy()).cuda(), short)
    assert (r.status, r.n_dirty, r.bytes) == exp == (0, 50, short)
    assert np.array_equal(reg.cpu().numpy(), reg_o) and np.array_equal(sh_t.cpu().numpy(), sh_o)
    ctx.shutdown()
