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


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_mixed_history(seed):
    rng = np.random.default_rng(seed)
    ctx = cc.Context()
    R = {}
    for rid, P, N in SPECS:
        cur = synth.raw_region(N, 1000 * seed + rid, "cuda")
        sh = ctx.register_region(rid, cur, P)
        h = cur.cpu().numpy().copy()
        n_pages = (N + P - 1) // P
        R[rid] = dict(P=P, N=N, n_pages=n_pages, cur=cur, sh=sh, hcur=h, hsh=h.copy(),
                      ver=np.zeros(n_pages, np.uint64), com=np.zeros(n_pages, np.uint64),
                      gver=torch.zeros(n_pages, dtype=torch.int64, device="cuda"),
                      gcom=torch.zeros(n_pages, dtype=torch.int64, device="cuda"), touched=set())
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

    def check_all():
        torch.cuda.synchronize()
        assert np.array_equal(log.cpu().numpy(), olog), "log differs"
        assert int(committed.item()) == W
        for rid, r in R.items():
            assert np.array_equal(r["sh"].cpu().numpy(), r["hsh"]), "shadow of region %d differs" % rid
            assert np.array_equal(r["gcom"].cpu().numpy().view(np.uint64), r["com"])

    ops = ["delta", "fused", "rle", "marked", "versions", "all", "snapshot", "reset"]
    weights = np.array([3, 3, 3, 4, 2, 2, 1, 1], dtype=float)
    for step in range(60):
        mutate()
        op = ops[int(rng.choice(len(ops), p=weights / weights.sum()))]
        rid = SPECS[int(rng.integers(0, 3))][0]
        r = R[rid]
        epoch = 100 + step
        res.clear()
        if op == "reset" or W > cap - (4 << 20):
            ctx.log_reset()
            W = 0
            torch.cuda.synchronize()
            continue
        if op == "delta":
            ctx.checkpoint_delta(rid, epoch, res)
            st, D, nb, W = oracle.checkpoint(r["hcur"], r["hsh"], r["P"], rid, epoch, olog, W)
            exp = (st, D.size, nb, W)
        elif op == "fused":
            ctx.checkpoint_delta_fused(rid, epoch, res)
            st, D, nb, W = oracle.checkpoint(r["hcur"], r["hsh"], r["P"], rid, epoch, olog, W)
            exp = (st, D.size, nb, W)
        elif op == "rle":
            rp = int(rng.choice([1, 2, 4, 16]))
            ctx.checkpoint_delta_rle(rid, epoch, rp, res)
            st, D, runs, nb, W = oracle.checkpoint_rle(r["hcur"], r["hsh"], r["P"], rid, epoch, rp, olog, W)
            exp = (st, D.size, nb, W)
        elif op == "marked":
            flags = int(rng.integers(0, 4))
            marks = sorted(set(list(r["touched"])[: int(rng.integers(0, 12))]) | set(rng.integers(0, r["n_pages"], 3).tolist()))
            bm = _bitmap(r["n_pages"], marks)
            gm = torch.from_numpy(bm.view(np.int32).copy()).cuda()
            ctx.checkpoint_marked(rid, epoch, gm, flags, res)
            st, D, nb, W = oracle.checkpoint_marked(r["hcur"], r["hsh"], r["P"], rid, epoch, bm, olog, W,
                                                    verify=bool(flags & 1), consume=bool(flags & 2))
            exp = (st, D.size, nb, W)
            torch.cuda.synchronize()
            assert np.array_equal(gm.cpu().numpy().view(np.uint32), bm)
        elif op == "versions":
            r["gver"].copy_(torch.from_numpy(r["ver"].view(np.int64).copy()))
            ctx.checkpoint_versions(rid, epoch, r["gver"], r["gcom"], res)
            st, D, nb, W = oracle.checkpoint_versions(r["hcur"], r["hsh"], r["P"], rid, epoch, r["ver"], r["com"], olog, W)
            exp = (st, D.size, nb, W)
        elif op == "all":
            ctx.checkpoint_all(epoch, res)
            st, ks, sts, kt, bt, W = oracle.checkpoint_all(oregs, epoch, olog, W)
            exp = (st, kt, bt, W)
            for x in R.values():
                x["touched"].clear()
        else:  # snapshot
            ctx.snapshot_region(rid, epoch, res)
            st, k, nb, W = oracle.snapshot(r["hcur"], r["hsh"], r["P"], rid, epoch, olog, W)
            exp = (st, k, nb, W)
        torch.cuda.synchronize()
        g = res.read()
        assert (g.status, g.n_dirty, g.bytes, g.log_offset_after) == exp, (step, op, rid, g.as_dict(), exp)
        assert g.status == 0
        if op in ("delta", "fused", "rle", "snapshot"):
            r["touched"].clear()
        if step % 10 == 9:
            check_all()
    check_all()
    # ---- compaction and replay of whatever the log holds now ----
    if W == 0:
        return
    ctx.apply_attach(20000)
    exp_out = np.zeros(cap, np.uint8)
    blank = [oracle.Region(rid, R[rid]["P"], np.zeros(R[rid]["N"], np.uint8)) for rid, _, _ in SPECS]
    st, nb, consumed, n_out = oracle.compact_log(olog, W, blank, exp_out)
    out = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    res.clear()
    ctx.compact_log(log, W, out, res)
    torch.cuda.synchronize()
    g = res.read()
    assert (g.status, g.n_dirty, g.bytes, g.log_offset_after) == (st, n_out, nb, consumed) and st == 0
    assert np.array_equal(out.cpu().numpy(), exp_out)
    for which, nbytes in ((log, W), (out, nb)):
        hosts = {rid: np.zeros(R[rid]["N"], np.uint8) for rid, _, _ in SPECS}
        e = oracle.apply_log(olog if which is log else exp_out, nbytes, [oracle.Region(rid, R[rid]["P"], hosts[rid]) for rid, _, _ in SPECS])
        for rid in R:
            R[rid]["cur"].zero_()
        res.clear()
        ctx.apply_log(which, nbytes, res)
        torch.cuda.synchronize()
        g = res.read()
        assert (g.status, g.n_dirty, g.bytes) == e and e[0] == 0
        for rid in R:
            assert np.array_equal(R[rid]["cur"].cpu().numpy(), hosts[rid])
    ctx.shutdown()
