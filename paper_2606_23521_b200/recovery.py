"""Recovery-side report (BASELINE.json configs[4], first half; SURVEY.md 8d "C5a", 8f #3):

    python -m paper_2606_23521_b200.recovery [--arena-gib 8] [--epochs 100] [--records 100]

Builds a committed log shaped like config 5a -- an arena registered as three regions with 4 / 16 / 64 KiB pages
(1/4, 1/4, 1/2 of the arena), `epochs` epochs of `records` page records each, epoch e on region (e mod 3)+1, pages
repeating across epochs -- with the library's own allocator-aware checkpoint (cc_checkpoint_marked on seeded page
sets; its log bytes are the ones the GPU tests prove bit-exact against the oracle), then times, with CUDA events:
  apply      cc_apply_log of that log, once from pinned host memory (host-link-bound) and once from device memory
  compact    cc_compact_log of that log (device -> device)
  snapshot   cc_snapshot_region of the 64 KiB-page region (every page -> log, device log)
Prints one JSON object.  No oracle involved.
"""
import argparse
import json
import statistics

import torch

from . import binding as cc

REGIONS = [(1, 0, 2, 4096), (2, 2, 2, 16384), (3, 4, 4, 65536)]      # id, offset/8, size/8, page bytes


def _ev(stream):
    e = torch.cuda.Event(enable_timing=True)
    e.record(stream)
    return e


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--arena-gib", type=float, default=8.0)
    ap.add_argument("--epochs", type=int, default=100)
    ap.add_argument("--records", type=int, default=100)
    ap.add_argument("--reps", type=int, default=5)
    a = ap.parse_args()
    dev = torch.device("cuda", 0)
    arena_bytes = int(a.arena_gib * 2**30) // (8 * 65536) * (8 * 65536)
    unit = arena_bytes // 8
    g = torch.Generator(device="cuda")
    g.manual_seed(1005)
    arena = torch.empty(arena_bytes, dtype=torch.uint8, device=dev)
    for o in range(0, arena_bytes, 1 << 28):
        n = min(1 << 28, arena_bytes - o)
        arena[o:o + n] = torch.randint(0, 256, (n,), dtype=torch.uint8, device=dev, generator=g)
    ctx = cc.Context(0)
    views = {}
    for rid, o8, s8, P in REGIONS:
        v = arena[o8 * unit:(o8 + s8) * unit]
        ctx.register_region(rid, v, P)
        views[rid] = (v, P, s8 * unit // P)
    n_rec = a.epochs * a.records
    cap = sum((16 + views[(e % 3) + 1][1]) * a.records + 32 for e in range(a.epochs))
    log_dev = torch.zeros(cap, dtype=torch.uint8, device=dev)
    ctx.log_attach(log_dev)
    ctx.apply_attach(n_rec + 256)
    res = cc.Result()
    stream = torch.cuda.current_stream()

    # ---- write the log: epoch e dirties `records` seeded pages of region (e mod 3)+1 ----
    cg = torch.Generator(device="cpu")
    cg.manual_seed(1005)
    last = {}
    for e in range(a.epochs):
        rid = (e % 3) + 1
        v, P, n_pages = views[rid]
        pages = torch.randperm(n_pages, generator=cg)[:a.records]
        if rid in last:
            pages[0] = last[rid]                          # a page repeats across epochs (last wins on replay)
        pages = torch.unique(pages)
        last[rid] = int(pages[0])
        pd = pages.to(dev)
        v.view(-1, P)[pd, :64] = torch.randint(0, 256, (pd.numel(), 64), dtype=torch.uint8, device=dev, generator=g)
        bm = torch.zeros((n_pages + 31) // 32, dtype=torch.int64)
        bm.index_put_((pages >> 5,), (1 << (pages & 31)), accumulate=True)
        marks = torch.where(bm >= 2**31, bm - 2**32, bm).to(torch.int32).to(dev)
        ctx.checkpoint_marked(rid, e + 1, marks, 0, res)
    torch.cuda.synchronize()
    r = res.read()
    assert r.status == 0
    W = int(r.log_offset_after)
    log_pin = torch.empty(W, dtype=torch.uint8, pin_memory=True)
    log_pin.copy_(log_dev[:W])
    torch.cuda.synchronize()

    def timed(fn, reps, before=None):
        ts = []
        for _ in range(reps + 1):
            if before:
                before()
            torch.cuda.synchronize()
            e0 = _ev(stream)
            fn()
            e1 = _ev(stream)
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return statistics.median(ts[1:]), min(ts[1:])

    out = {"config": {"arena_GiB": arena_bytes / 2**30, "regions": "4 / 16 / 64 KiB pages on 1/4, 1/4, 1/2 of the arena",
                      "epochs": a.epochs, "page_records": None, "log_bytes": W}}

    # ---- apply ----
    def scramble():
        for rid, (v, P, n_pages) in views.items():
            v.view(-1, P)[:, :64] = 0                     # every page differs from the logged bytes again
    for name, lg in (("apply_from_pinned_host_log", log_pin), ("apply_from_pinned_host_log_staged", log_pin),
                     ("apply_from_device_log", log_dev)):
        ctx.apply_stage_attach(W if name.endswith("staged") else 0)      # staged: one DMA pass over the host link
        med, best = timed(lambda: ctx.apply_log(lg, W, res), a.reps, scramble)
        rr = res.read()
        assert rr.status == 0 and rr.bytes == W, rr.as_dict()
        out[name] = {"ms": round(med, 4), "best_ms": round(best, 4), "records": int(rr.n_dirty),
                     "records_per_s": round(rr.n_dirty / (med * 1e-3)), "log_GBps": round(W / (med * 1e-3) / 1e9, 2)}
    ctx.apply_stage_attach(0)
    out["config"]["page_records"] = int(rr.n_dirty)
    # ---- compact ----
    out_log = torch.zeros(W, dtype=torch.uint8, device=dev)
    med, best = timed(lambda: ctx.compact_log(log_dev, W, out_log, res), a.reps)
    rr = res.read()
    assert rr.status == 0, rr.as_dict()
    out["compact_device_to_device"] = {"ms": round(med, 4), "best_ms": round(best, 4), "records_in": out["config"]["page_records"],
                                       "records_out": int(rr.n_dirty), "bytes_out": int(rr.bytes),
                                       "input_GBps": round(W / (med * 1e-3) / 1e9, 2)}
    # replay of the compacted log == replay of the original
    scramble()
    ctx.apply_log(log_dev, W, res)
    torch.cuda.synchronize()
    ref = arena.clone()
    scramble()
    ctx.apply_log(out_log, int(rr.bytes), res)
    torch.cuda.synchronize()
    assert res.read().status == 0 and torch.equal(ref, arena), "compacted log replays differently"
    del ref
    # ---- base snapshot of the 64 KiB-page region ----
    v, P, n_pages = views[3]
    snap_cap = n_pages * (16 + P) + 32
    free, _ = torch.cuda.mem_get_info()
    if free > snap_cap + (2 << 30):
        snap = torch.empty(snap_cap, dtype=torch.uint8, device=dev)
        ctx.log_attach(snap)
        med, best = timed(lambda: ctx.snapshot_region(3, 999, res), a.reps, lambda: ctx.log_reset())
        rr = res.read()
        assert rr.status == 0 and rr.n_dirty == n_pages
        nb = n_pages * P
        out["snapshot_region_device_log"] = {"ms": round(med, 4), "best_ms": round(best, 4), "pages": n_pages,
                                             "region_GBps": round(nb / (med * 1e-3) / 1e9, 1),
                                             "hbm_GBps_3x": round(3 * nb / (med * 1e-3) / 1e9, 1)}
    ctx.shutdown()
    print(json.dumps(out))


if __name__ == "__main__":
    main()
