"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

C2 (8 GiB KV cache) is checked element by element against the oracle (the host has room);
C4 (64 GiB) is checked chunk-wise: dirty list against the oracle's scan of every chunk, every log
record against the oracle's CRC + the live bytes; C5a (8 GiB arena, 10,000-record log) against
oracle_apply on a host copy; C5b (10,000 ring tasks) with bit-exact logs on the first tasks and
closed-form k on all.  Tests skip when the device or host is too small.
"""
import struct

import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc
from gpu_util import gpu_checkpoint, verify_all_dirty

pytestmark = pytest.mark.gpu


def _need(dev_gib, host_gib=0):
    free, _ = torch.cuda.mem_get_info()
    if free < dev_gib * 2**30:
        pytest.skip("needs %d GiB of free device memory" % dev_gib)
    if host_gib:
        import psutil
        if psutil.virtual_memory().available < host_gib * 2**30:
            pytest.skip("needs %d GiB of host memory" % host_gib)


def test_c2_full_8gib_kv_cache():
    _need(20, 20)
    P, layers, blocks, seqs = 65536, 32, 4096, 256
    cur = synth.kv_cache_region(layers, blocks, 1002, "cuda")
    assert cur.numel() == 8 << 30
    ctx = cc.Context()
    shadow = ctx.register_region(1, cur, P)
    old_h = cur.cpu().numpy()                       # == shadow
    pages = synth.kv_decode_step(cur, layers, blocks, seqs, 1002)
    assert len(pages) == 8192
    nb_exp = 8192 * (16 + P) + 32
    assert nb_exp == 537_002_016                    # closed form, SURVEY.md 8c
    log = torch.zeros(nb_exp, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    r = gpu_checkpoint(ctx, 1, 77)
    assert (r.status, r.n_dirty, r.bytes) == (0, 8192, nb_exp)
    cur_h = cur.cpu().numpy()
    olog = np.zeros(nb_exp, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur_h, old_h, P, 1, 77, olog, 0)        # old_h becomes the oracle's new shadow
    assert st == 0 and D.tolist() == pages.tolist() == ctx.dirty_list(1).tolist()
    assert np.array_equal(log.cpu().numpy(), olog)
    assert torch.equal(shadow, cur) and np.array_equal(old_h, cur_h)
    r = gpu_checkpoint(ctx, 1, 78)
    assert r.n_dirty == 0 and r.bytes == 0


def _equal_chunked(a, b, chunk=1 << 30):
    return all(torch.equal(a[o:o + chunk], b[o:o + chunk]) for o in range(0, a.numel(), chunk))


def test_c4_full_64gib_sparse_page_size_sweep():
    """Config 4, sparse sweep: ONE 64 GiB region, 0.1 % of its 4 KiB pages flipped; the same memory is
    registered three times (P = 4, 16, 64 KiB).  Dirty lists of all three against the oracle's scan of every
    4 GiB chunk; then a full checkpoint at P = 64 KiB with every record checked against the oracle's CRC."""
    _need(140, 12)
    N = 64 << 30
    cur = synth.bf16_normal_region(N, 1004, "cuda")
    shadow = torch.empty_like(cur)
    for o in range(0, N, 1 << 30):
        shadow[o:o + (1 << 30)] = cur[o:o + (1 << 30)]
    Ps = (4096, 16384, 65536)
    ctx = cc.Context()
    for i, P in enumerate(Ps):
        ctx.register_region(i + 1, cur, P, shadow=shadow, snapshot_now=False)
    pages4k, offs, masks = synth.sparse_xor_flips(cur, 4096, 0.001, 1004)
    assert len(pages4k) == -(-(N // 4096) // 1000) == 16778
    # oracle: chunk-wise scans at the three page sizes
    chunk = 4 << 30
    D_or = {P: [] for P in Ps}
    for o in range(0, N, chunk):
        c = cur[o:o + chunk].cpu().numpy()
        s = shadow[o:o + chunk].cpu().numpy()
        for P in Ps:
            D_or[P].append(np.nonzero(oracle.scan_mt(c, s, P, 16))[0] + o // P)
        del c, s
    D_or = {P: np.concatenate(v) for P, v in D_or.items()}
    assert D_or[4096].tolist() == pages4k.tolist()
    res = cc.Result()
    for i, P in enumerate(Ps):
        res.clear()
        ctx.scan_only(i + 1, res)
        torch.cuda.synchronize()
        assert res.read().n_dirty == D_or[P].size
        assert ctx.dirty_list(i + 1).tolist() == D_or[P].tolist(), P
    # full checkpoint at 64 KiB pages
    P = 65536
    k = D_or[P].size
    log = torch.zeros(k * (16 + P) + 32, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    r = gpu_checkpoint(ctx, 3, 5)
    assert (r.status, r.n_dirty, r.bytes) == (0, k, k * (16 + P) + 32)
    lg = log.cpu().numpy()
    step = 16 + P
    for i in range(0, k, 3):
        rid, pi, ln, crc = struct.unpack_from("<IIII", lg, i * step)
        assert (rid, pi, ln) == (3, int(D_or[P][i]), P)
        page = cur[pi * P:(pi + 1) * P].cpu().numpy()
        assert np.array_equal(lg[i * step + 16:(i + 1) * step], page)
        assert crc == oracle.crc32c(page)
    cp = lg[k * step:]
    assert struct.unpack("<IIII", cp[:16].tobytes())[:3] == (0xFFFFFFFF, 0xFFFFFFFF, 16)
    assert struct.unpack("<QII", cp[16:].tobytes()) == (5, 3, k)
    assert struct.unpack_from("<I", cp, 12)[0] == oracle.crc32c(cp[16:])
    assert _equal_chunked(shadow, cur)
    r = gpu_checkpoint(ctx, 1, 6)                      # the 4 KiB registration now sees a clean region
    assert r.n_dirty == 0


def test_c4_all_dirty_4gib_device_log():
    """100 % dirty (gather-bound worst case) at a size whose log fits beside the region."""
    _need(16, 10)
    P, N = 16384, 4 << 30
    cur = synth.bf16_normal_region(N, 1004, "cuda")
    ctx = cc.Context()
    shadow = ctx.register_region(1, cur, P)
    pages, offs, masks = synth.sparse_xor_flips(cur, P, 1.0, 99)
    n_pages = N // P
    log = torch.zeros(n_pages * (16 + P) + 32, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    r = gpu_checkpoint(ctx, 1, 6)
    assert (r.status, r.n_dirty, r.bytes) == (0, n_pages, log.numel())
    # all pages dirty => payloads concatenated == region (north_star invariant), headers in order
    body = log[:n_pages * (16 + P)].view(n_pages, 16 + P)
    assert torch.equal(body[:, 16:], cur.view(n_pages, P))
    hdr = body[:, :16].contiguous().view(torch.int32).view(n_pages, 4)
    assert torch.equal(hdr[:, 1].to(torch.int64), torch.arange(n_pages, device="cuda"))
    assert bool((hdr[:, 0] == 1).all()) and bool((hdr[:, 2] == P).all())
    # CRCs of a sample of records against the oracle
    lg_crc = hdr[:, 3].cpu().numpy().view(np.uint32)
    for i in list(range(0, n_pages, 4099)) + [n_pages - 1]:
        assert int(lg_crc[i]) == oracle.crc32c(cur[i * P:(i + 1) * P].cpu().numpy())
    assert torch.equal(shadow, cur)


def test_c5a_full_recovery_10000_records():
    _need(20, 20)
    arena_bytes = 8 << 30
    arena = synth.raw_region(arena_bytes, 1005, "cuda")
    unit = arena_bytes // 8
    eps = synth.recovery_epochs(arena_bytes, 100, 100, 1005, forced_repeats=50)
    n_rec = sum(e.pages.numel() for e in eps)
    cap = sum(e.payloads.numel() + 16 * e.pages.numel() + 32 for e in eps)
    assert n_rec >= 9_950 and cap > 280_000_000
    olog = np.zeros(cap, dtype=np.uint8)
    views = {rid: (o8 * unit, s8 * unit, P) for rid, o8, s8, P in synth.C5A_REGIONS}
    W = 0
    for e in eps:
        o, sz, P = views[e.region_id]
        st, W = oracle.write_epoch(olog, W, e.region_id, e.epoch, sz, P, e.pages.numpy(), e.payloads.numpy())
        assert st == 0
    host = arena.cpu().numpy()
    exp = oracle.apply_log(olog, W, [oracle.Region(rid, P, host[o:o + sz]) for rid, (o, sz, P) in views.items()])
    assert exp == (0, n_rec, W)
    for pinned in (True, False):
        work = arena.clone()
        ctx = cc.Context()
        for rid, (o, sz, P) in views.items():
            ctx.register_region(rid, work[o:o + sz], P)
        ctx.apply_attach(n_rec + 128)
        lt = torch.from_numpy(olog)
        lt = lt.pin_memory() if pinned else lt.cuda()
        res = cc.Result()
        ctx.apply_log(lt, W, res)
        torch.cuda.synchronize()
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes, r.epoch) == (0, n_rec, W, 100)
        assert all(np.array_equal(work[o:o + (1 << 30)].cpu().numpy(), host[o:o + (1 << 30)])
                   for o in range(0, arena_bytes, 1 << 30))
        ctx.shutdown()
        del work


def test_c5b_full_10000_ring_tasks():
    _need(2)
    P, n_pages, n_mut, n_tasks = 4096, 65536, 656, 10_000
    cur = synth.raw_region(P * n_pages, 1006, "cuda")
    ctx = cc.Context(ring_capacity=256, max_lifetime_ns=int(120e9))
    sh = ctx.register_region(1, cur, P)
    per = n_mut * (16 + P) + 32
    assert per == 2_697_504                                  # closed form, SURVEY.md 8c
    log = torch.zeros(1 << 30, dtype=torch.uint8, pin_memory=True)
    ctx.log_attach(log)
    host_cur = cur.cpu().numpy().copy()
    host_sh = host_cur.copy()
    A = 2 * ((1006 * 7919 + 12345) % 100000) + 1
    n_parity = 64
    olog = np.zeros(n_parity * per, dtype=np.uint8)
    W = 0
    ctx.worker_start()
    try:
        ck = []
        for t in range(n_tasks):
            if t and t % 256 == 0:
                ctx.wait(ck[-1], 30.0)
                if t == 256:
                    assert np.array_equal(log.numpy()[:n_parity * per], olog)
                ctx.submit(cc.CC_TASK_LOG_RESET)
            pages, h = synth.worker_mutation_pages(t, n_pages, n_mut, 1006)
            while True:
                try:
                    ctx.submit(cc.CC_TASK_TEST_MUTATE, region_id=1, arg0=n_mut, arg1=A, arg2=h)
                    break
                except cc.ConcordiaError as e:
                    assert e.code == cc.CC_ERR_RING_FULL
            while True:
                try:
                    ck.append(ctx.submit(cc.CC_TASK_DELTA_CKPT, region_id=1, epoch=t))
                    break
                except cc.ConcordiaError as e:
                    assert e.code == cc.CC_ERR_RING_FULL
            if t < n_parity:
                assert len(set(pages)) == n_mut
                for j, p in enumerate(pages):
                    host_cur[p * P + (h + j) % P] ^= 0x5A
                st, D, nb, W = oracle.checkpoint(host_cur, host_sh, P, 1, t, olog, W)
                assert st == 0 and D.size == n_mut
            if len(ck) >= 100:                                # 100 checkpoints = ~200 submissions back: slot not yet reused
                s = ck[len(ck) - 100]
                r = ctx.poll(s) or ctx.wait(s, 30.0)
                assert (r.status, r.n_dirty, r.bytes) == (0, n_mut, per), (s, r.as_dict())
        r = ctx.wait(ck[-1], 30.0)
        assert (r.status, r.n_dirty, r.bytes) == (0, n_mut, per)
        h, t = ctx.peek_queue()
        assert h == t
    finally:
        ctx.worker_stop()
    torch.cuda.synchronize()
    assert torch.equal(sh, cur)
    ctx.shutdown()


@pytest.mark.parametrize("P", [4096, 16384, 65536])
def test_c4_full_32gib_all_dirty_every_record_against_the_oracle(P):
    """Config 4, 100 % dirty leg AT THE MEASURED SIZE: 32 GiB (the largest slice whose device log fits beside region
    and shadow, SURVEY.md 8d fallback ii), every page dirty, at 4 / 16 / 64 KiB pages.  EVERY record of the 32 GiB
    device log -- header, CRC32C, payload -- and the commit record are compared with oracle.checkpoint run on every
    1 GiB chunk of the region (oracle/chunked.py); shadow == region afterwards."""
    _need(100, 60)
    N = 32 << 30
    cur = synth.bf16_normal_region(N, 1004, "cuda")
    ctx = cc.Context()
    shadow = ctx.register_region(1, cur, P)
    n_pages = N // P
    log = torch.empty(n_pages * (16 + P) + 32, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    offs, masks = synth.all_dirty_flips(N, P, 1004 + P, "cuda")
    synth.toggle_flips(cur, offs, masks)
    r = gpu_checkpoint(ctx, 1, 6)
    assert (r.status, r.n_dirty, r.bytes) == (0, n_pages, log.numel())
    k, nb, D = verify_all_dirty(cur, log, offs, masks, P, 1, 6)
    assert (k, nb) == (n_pages, log.numel())
    assert _equal_chunked(shadow, cur)
    r = gpu_checkpoint(ctx, 1, 7)
    assert r.n_dirty == 0 and r.bytes == 0
    ctx.shutdown()


@pytest.mark.parametrize("P", [4096, 16384, 65536])
def test_c4_full_64gib_arena_as_8_regions_through_one_pinned_log(P):
    """SURVEY.md 8d capacity fallback (i), BASELINE.json configs[3] "100 % pages dirty ... sweeping page size over
    4/16/64 KiB": the 64 GiB arena registered as 8 x 8 GiB regions, every page dirty, each checkpointed into ONE pinned
    8.0-8.1 GiB host log; every record of every region (16.8 M records in all at 4 KiB pages) is checked against the
    oracle chunk-wise, the shadows against the regions, and the log is rewound between regions."""
    _need(140, 40)
    R, regions = 8 << 30, 8
    arena = synth.bf16_normal_region(regions * R, 1004, "cuda")
    ctx = cc.Context()
    shadows = [ctx.register_region(i + 1, arena[i * R:(i + 1) * R], P) for i in range(regions)]
    n_pages = R // P
    cap = n_pages * (16 + P) + 32
    hlog = torch.empty(cap, dtype=torch.uint8, pin_memory=True)
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(hlog, committed)
    for i in range(regions):
        v = arena[i * R:(i + 1) * R]
        offs, masks = synth.all_dirty_flips(R, P, 7000 + i, "cuda")
        synth.toggle_flips(v, offs, masks)
        r = gpu_checkpoint(ctx, i + 1, i)
        assert (r.status, r.n_dirty, r.bytes, int(committed.item())) == (0, n_pages, cap, cap), r.as_dict()
        kk, nb, D = verify_all_dirty(v, hlog, offs, masks, P, i + 1, i, log_is_host=True)
        assert (kk, nb) == (n_pages, cap) and _equal_chunked(shadows[i], v)
        ctx.log_reset()
    ctx.shutdown()


@pytest.mark.parametrize("R", [3, 5])
def test_single_pass_run_records_16gib_region_odd_run_length(R):
    """16 GiB at 4 KiB pages (2^22 + 3 pages) with a run length that is no power of two, forced onto the single pass: the
    tile size has a lower bound of ceil(n_pages / 2^20) pages (the look-back table has 2^20 words) that rounding to a
    multiple of run_pages must not undercut -- rounded DOWN, 4 -> 3 pages gave 1.4 M tiles and writes past the workspace.
    Mostly-zero contents (the host copies stay virtual); the dirty pages carry seeded bytes."""
    _need(36, 12)
    P, n_pages = 4096, (1 << 22) + 3
    N = n_pages * P
    rng = np.random.default_rng(160 + R)
    starts = rng.choice(n_pages - 16, 2000, replace=False)
    pages = np.unique(np.concatenate([starts + j for j in range(R + 2)] + [np.array([0, n_pages - 2, n_pages - 1])]))
    idx = pages * P + rng.integers(0, P, pages.size)
    vals = rng.integers(1, 256, pages.size).astype(np.uint8)
    cur = torch.zeros(N, dtype=torch.uint8, device="cuda")
    shadow = torch.zeros(N, dtype=torch.uint8, device="cuda")
    cur[torch.from_numpy(idx).cuda()] = torch.from_numpy(vals).cuda()
    cur_h, sh_h = np.zeros(N, np.uint8), np.zeros(N, np.uint8)
    cur_h[idx] = vals
    cap = pages.size * (16 + P) + 4096
    olog = np.zeros(cap, np.uint8)
    st, D, runs, nb, W = oracle.checkpoint_rle(cur_h, sh_h, P, 4, 9, R, olog, 0)
    assert st == 0 and D.tolist() == pages.tolist() and 0 < runs < pages.size
    ctx = cc.Context()
    ctx.register_region(4, cur, P, shadow=shadow, snapshot_now=False)
    glog = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    ctx.log_attach(glog)
    res = cc.Result()
    ctx.checkpoint_ex(4, 9, res, path=cc.CC_PATH_SINGLE_PASS, run_pages=R)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (0, D.size, nb, W), r.as_dict()
    assert ctx.dirty_list(4).tolist() == D.tolist()
    assert np.array_equal(glog.cpu().numpy(), olog)
    assert _equal_chunked(shadow, cur)                      # every dirty page refreshed, nothing else touched
    ctx.shutdown()


def test_replay_of_a_base_snapshot_larger_than_64gib():
    """PAPER.md:L227 "replays the latest base snapshot and committed AOF suffix" at config 4's own size: the base
    snapshot of a 64 GiB region (64 KiB pages, allocator-aware: no shadow) is a 64.016 GiB log -- more than 2^36 bytes,
    so its commit record lies beyond what the parallel parse's 32-bit candidate offsets reach and the whole log takes
    the serial parser.  Too large for the host oracle in one piece, so: result fields against the closed form; every
    header field and every payload byte against the region on the device (exact); the CRC32C of sampled records
    (first, middle, the first one past 2^36, last) and the commit record against the oracle; then the region is zeroed
    and replayed from the log and must equal the payloads again; finally one flipped payload byte in the LAST record
    (past 2^36) must give CC_ERR_CORRUPT with nothing applied (single epoch)."""
    _need(136, 4)
    P, N = 65536, 64 << 30
    n_pages = N // P
    nbytes = n_pages * (16 + P) + 32
    assert nbytes > (1 << 36)
    region = synth.bf16_normal_region(N, 2036, "cuda")
    ctx = cc.Context()
    ctx.register_region(9, region, P, no_shadow=True)
    log = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    ctx.apply_attach(n_pages + 64)
    res = cc.Result()
    ctx.snapshot_region(9, 41, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch) == (0, n_pages, nbytes, nbytes, 41), r.as_dict()
    recs = log[:n_pages * (16 + P)].view(n_pages, 16 + P)
    step = 16384                                                    # pages per 1 GiB chunk

    def region_equals_payloads():
        return all(torch.equal(recs[a:a + step, 16:], region[a * P:(a + step) * P].view(-1, P)) for a in range(0, n_pages, step))

    assert region_equals_payloads()
    hdr = recs[:, :16].contiguous().view(torch.int32).view(n_pages, 4)
    assert bool((hdr[:, 0] == 9).all()) and bool((hdr[:, 2] == P).all())
    assert torch.equal(hdr[:, 1], torch.arange(n_pages, dtype=torch.int32, device="cuda"))
    past = (1 << 36) // (16 + P) + 1                                # first record that starts beyond 2^36 bytes
    assert past < n_pages
    for i in (0, 1, n_pages // 2, past, n_pages - 1):
        page = region[i * P:(i + 1) * P].cpu().numpy()
        assert int(hdr[i, 3].item()) & 0xFFFFFFFF == oracle.crc32c(page), i
    tail = log[nbytes - 32:].cpu().numpy().tobytes()
    cid, cid2, clen, ccrc, epoch, rid, k = struct.unpack("<IIIIQII", tail)
    assert (cid, cid2, clen, epoch, rid, k) == (0xFFFFFFFF, 0xFFFFFFFF, 16, 41, 9, n_pages)
    assert ccrc == oracle.crc32c(np.frombuffer(tail[16:], np.uint8))
    # replay into the zeroed region
    region.zero_()
    res.clear()
    ctx.apply_log(log, nbytes, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.epoch) == (0, n_pages, nbytes, 1), r.as_dict()
    assert region_equals_payloads()
    # damage the last record (its bytes lie past 2^36): the only epoch fails its check, nothing is applied
    region.zero_()
    log[nbytes - 32 - 100] ^= 0x20
    res.clear()
    ctx.apply_log(log, nbytes, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes, r.epoch) == (cc.CC_ERR_CORRUPT, 0, 0, 0), r.as_dict()
    assert not any(bool(region[o:o + (1 << 30)].any()) for o in range(0, N, 1 << 30))
    ctx.shutdown()
