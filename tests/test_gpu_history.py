"""GPU parity under a long MIXED history: a seeded random sequence of every checkpoint flavour (three-kernel, fused,
run-length, allocator-aware trusted / verified / consumed, version counters, all-regions, base snapshot), log resets,
mutations, and at the end compaction and replay -- on three regions of different page sizes sharing one log, each step
checked against the oracle (result fields), the whole log / shadows / marks / version tables checked bit for bit at
checkpoints along the way.  Catches state leaking from one path into the next (bitmaps, tickets, look-back tags,
per-record CRC words, plan fields)."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc

pytestmark = pytest.mark.gpu

SPECS = [(3, 4096, 4096 * 300 - 2048), (8, 65536, 65536 * 24), (5, 256, 256 * 2000 - 64)]


def _bitmap(n_pages, pages):
    bm = np.zeros((n_pages + 31) // 32, dtype=np.uint32)
    for p in pages:
        bm[p >> 5] |= np.uint32(1 << (p & 31))
    return bm


@pytest.mark.parametrize("seed,worker", [(1, False), (2, False), (3, False), (4, True), (5, True)])
def test_mixed_history(seed, worker):
    """worker=True: the same history submitted as tasks to the persistent worker (16 CTAs, so that the test's own torch
    kernels -- the "application" -- run beside it); no device-wide synchronisation while it is resident."""
    rng = np.random.default_rng(seed)
    ctx = cc.Context(ring_capacity=16, worker_blocks=16, max_lifetime_ns=int(120e9)) if worker else cc.Context()
    sync = (lambda: torch.cuda.current_stream().synchronize()) if worker else torch.cuda.synchronize
    R = {}
    for rid, P, N in SPECS:
        cur = synth.raw_region(N, 1000 * seed + rid, "cuda")
        sh = ctx.register_region(rid, cur, P)
        h = cur.cpu().numpy().copy()
        n_pages = (N + P - 1) // P
        R[rid] = dict(P=P, N=N, n_pages=n_pages, cur=cur, sh=sh, hcur=h, hsh=h.copy(),
                      ver=np.zeros(n_pages, np.uint64), com=np.zeros(n_pages, np.uint64),
                      gver=torch.zeros(n_pages, dtype=torch.int64, device="cuda"),
                      gcom=torch.zeros(n_pages, dtype=torch.int64, device="cuda"),
                      gm=torch.zeros((n_pages + 31) // 32, dtype=torch.int32, device="cuda"), touched=set())
        cur[0] ^= 0                                    # warm torch's allocator for the small temporaries of mutate()
    cap = 24 << 20
    pinned = seed % 2 == 0
    log = torch.zeros(cap, dtype=torch.uint8, pin_memory=True) if pinned else torch.zeros(cap, dtype=torch.uint8, device="cuda")
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(log, committed)
    olog = np.zeros(cap, np.uint8)
    W = 0
    res = cc.Result()
    oregs = [oracle.Region(rid, R[rid]["P"], R[rid]["hcur"], R[rid]["hsh"]) for rid, _, _ in SPECS]

    def mutate():
        for _ in range(int(rng.integers(1, 4))):
            r = R[SPECS[int(rng.integers(0, 3))][0]]
            a = int(rng.integers(0, r["n_pages"]))
            for p in range(a, min(r["n_pages"], a + int(rng.integers(1, 6)))):
                off = p * r["P"] + int(rng.integers(0, min(r["P"], r["N"] - p * r["P"])))
                r["hcur"][off] ^= 0x6D
                r["cur"][off] ^= 0x6D
                r["ver"][p] += np.uint64(1)
                r["touched"].add(p)

    def run(kind, host_call, **task):
        """host-launched call, or the equivalent task through the ring; returns the result record"""
        sync()
        if worker:
            return ctx.wait(ctx.submit(kind, **task), 30.0)
        res.clear()
        host_call()
        torch.cuda.synchronize()
        return res.read()

    def check_all():
        sync()
        assert np.array_equal(log.cpu().numpy(), olog), "log differs"
        assert int(committed.item()) == W
        for rid, r in R.items():
            assert np.array_equal(r["sh"].cpu().numpy(), r["hsh"]), "shadow of region %d differs" % rid
            assert np.array_equal(r["gcom"].cpu().numpy().view(np.uint64), r["com"])

    ctx.apply_attach(20000)
    out = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    if worker:
        torch.cuda.synchronize()
        ctx.worker_start()
    ops = ["delta", "fused", "rle", "marked", "versions", "all", "snapshot", "reset"]
    weights = np.array([3, 3, 3, 4, 2, 2, 1, 1], dtype=float)
    for step in range(60):
        mutate()
        op = ops[int(rng.choice(len(ops), p=weights / weights.sum()))]
        rid = SPECS[int(rng.integers(0, 3))][0]
        r = R[rid]
        epoch = 100 + step
        if op == "reset" or W > cap - (4 << 20):
            run(cc.CC_TASK_LOG_RESET, ctx.log_reset)
            W = 0
            continue
        if op == "delta":
            g = run(cc.CC_TASK_DELTA_CKPT, lambda: ctx.checkpoint_delta(rid, epoch, res), region_id=rid, epoch=epoch)
            st, D, nb, W = oracle.checkpoint(r["hcur"], r["hsh"], r["P"], rid, epoch, olog, W)
            exp = (st, D.size, nb, W)
        elif op == "fused":
            g = run(cc.CC_TASK_DELTA_CKPT, lambda: ctx.checkpoint_delta_fused(rid, epoch, res), region_id=rid, epoch=epoch,
                    flags=cc.CC_TASKF_FUSED)
            st, D, nb, W = oracle.checkpoint(r["hcur"], r["hsh"], r["P"], rid, epoch, olog, W)
            exp = (st, D.size, nb, W)
        elif op == "rle":
            rp = int(rng.choice([1, 2, 4, 16]))
            g = run(cc.CC_TASK_DELTA_CKPT, lambda: ctx.checkpoint_delta_rle(rid, epoch, rp, res), region_id=rid, epoch=epoch,
                    flags=cc.CC_TASKF_RLE, arg0=rp)
            st, D, runs, nb, W = oracle.checkpoint_rle(r["hcur"], r["hsh"], r["P"], rid, epoch, rp, olog, W)
            exp = (st, D.size, nb, W)
        elif op == "marked":
            flags = int(rng.integers(0, 4))
            marks = sorted(set(list(r["touched"])[: int(rng.integers(0, 12))]) | set(rng.integers(0, r["n_pages"], 3).tolist()))
            bm = _bitmap(r["n_pages"], marks)
            gm = r["gm"]                                  # allocated before the worker went resident
            gm.copy_(torch.from_numpy(bm.view(np.int32).copy()))
            g = run(cc.CC_TASK_MARKED_CKPT, lambda: ctx.checkpoint_marked(rid, epoch, gm, flags, res), region_id=rid, epoch=epoch,
                    arg0=gm.data_ptr(), arg1=flags)
            st, D, nb, W = oracle.checkpoint_marked(r["hcur"], r["hsh"], r["P"], rid, epoch, bm, olog, W,
                                                    verify=bool(flags & 1), consume=bool(flags & 2))
            exp = (st, D.size, nb, W)
            sync()
            assert np.array_equal(gm.cpu().numpy().view(np.uint32), bm)
        elif op == "versions":
            r["gver"].copy_(torch.from_numpy(r["ver"].view(np.int64).copy()))
            g = run(cc.CC_TASK_VERSION_CKPT, lambda: ctx.checkpoint_versions(rid, epoch, r["gver"], r["gcom"], res), region_id=rid,
                    epoch=epoch, arg0=r["gver"].data_ptr(), arg1=r["gcom"].data_ptr())
            st, D, nb, W = oracle.checkpoint_versions(r["hcur"], r["hsh"], r["P"], rid, epoch, r["ver"], r["com"], olog, W)
            exp = (st, D.size, nb, W)
        elif op == "all":
            g = run(cc.CC_TASK_CKPT_ALL, lambda: ctx.checkpoint_all(epoch, res), epoch=epoch)
            st, ks, sts, kt, bt, W = oracle.checkpoint_all(oregs, epoch, olog, W)
            exp = (st, kt, bt, W)
            for x in R.values():
                x["touched"].clear()
        else:  # snapshot
            g = run(cc.CC_TASK_SNAPSHOT, lambda: ctx.snapshot_region(rid, epoch, res), region_id=rid, epoch=epoch)
            st, k, nb, W = oracle.snapshot(r["hcur"], r["hsh"], r["P"], rid, epoch, olog, W)
            exp = (st, k, nb, W)
        assert (g.status, g.n_dirty, g.bytes, g.log_offset_after) == exp, (step, op, rid, g.as_dict() if hasattr(g, "as_dict") else g, exp)
        assert g.status == 0
        if op in ("delta", "fused", "rle", "snapshot"):
            r["touched"].clear()
        if step % 10 == 9:
            check_all()
    check_all()
    # ---- compaction and replay of whatever the log holds now ----
    if W == 0:
        if worker:
            ctx.worker_stop()
        ctx.shutdown()
        return
    exp_out = np.zeros(cap, np.uint8)
    blank = [oracle.Region(rid, R[rid]["P"], np.zeros(R[rid]["N"], np.uint8)) for rid, _, _ in SPECS]
    st, nb, consumed, n_out = oracle.compact_log(olog, W, blank, exp_out)
    g = run(cc.CC_TASK_COMPACT_LOG, lambda: ctx.compact_log(log, W, out, res), arg0=log.data_ptr(), arg1=W, arg2=out.data_ptr(),
            arg3=out.numel())
    assert (g.status, g.n_dirty, g.bytes, g.log_offset_after) == (st, n_out, nb, consumed) and st == 0
    assert np.array_equal(out.cpu().numpy(), exp_out)
    for which, nbytes in ((log, W), (out, nb)):
        hosts = {rid: np.zeros(R[rid]["N"], np.uint8) for rid, _, _ in SPECS}
        e = oracle.apply_log(olog if which is log else exp_out, nbytes, [oracle.Region(rid, R[rid]["P"], hosts[rid]) for rid, _, _ in SPECS])
        for rid in R:
            R[rid]["cur"].zero_()
        g = run(cc.CC_TASK_RESTORE, lambda: ctx.apply_log(which, nbytes, res), arg0=which.data_ptr(), arg1=nbytes)
        assert (g.status, g.n_dirty, g.bytes) == e and e[0] == 0
        sync()
        for rid in R:
            assert np.array_equal(R[rid]["cur"].cpu().numpy(), hosts[rid])
    if worker:
        ctx.worker_stop()
    ctx.shutdown()
