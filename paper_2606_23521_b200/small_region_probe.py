"""Timeline of a small-region checkpoint (c1 / c3) per path, with the trace build (-DCC_TRACE_ON=1)."""
import ctypes, statistics, sys, os
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import torch
import synth
import paper_2606_23521_b200 as cc

dev = torch.device("cuda:0")
flushbuf = torch.empty(512 << 20, dtype=torch.uint8, device=dev)

def run(name, path, cold, host_log=False, n=12):
    if name == "c1":
        P = 4096
        cur = synth.raw_region(64 << 20, 1001, dev); old = cur.clone()
        pages = synth.mutate_byte_flips(cur, P, 0.01, 1001)
    else:
        P = 65536
        cur = synth.lora_region(32, 1003, dev); old = cur.clone()
        pages = synth.lora_update(cur, P, 0.05, 1003)
    N = cur.numel(); k = len(pages)
    ctx = cc.Context(0)
    shadow = ctx.register_region(1, cur, P, shadow=cur.clone(), snapshot_now=False)
    cap = (N // P) * (16 + P) + 32
    log = torch.zeros(cap, dtype=torch.uint8, pin_memory=True) if host_log else torch.zeros(cap, dtype=torch.uint8, device=dev)
    ctx.log_attach(log)
    res = cc.Result()
    pg = pages.to(dev)
    offs = pg * P + (pg * 2654435761 % P)
    masks = torch.full((k,), 0x11, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    ev, dv, tr = [], [], []
    tbuf = (ctypes.c_uint64 * 32)()
    for it in range(n):
        synth.toggle_flips(cur, offs, masks)
        if cold:
            flushbuf.fill_(it & 0xFF)
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        torch.cuda._sleep(300000)
        e0.record(stream)
        ctx.checkpoint_ex(1, it, res, path=path)
        e1.record(stream)
        torch.cuda.synchronize()
        r = res.read()
        assert r.status == 0 and r.n_dirty == k
        ctx.lib.cc_debug_trace(ctx.h, tbuf)
        ctx.log_reset()
        if it >= 3:
            ev.append(e0.elapsed_time(e1) * 1e3)
            dv.append((r.t_end_ns - r.t_start_ns) / 1e3)
            t0 = r.t_start_ns
            tr.append([(int(tbuf[i]) - t0) / 1e3 if tbuf[i] else None for i in range(16)])
    med = lambda xs: statistics.median(xs)
    names = {0: "scan0", 1: "scan1(b0)", 2: "compact0", 3: "compact1", 4: "gather0", 5: "items0", 9: "items1(b0)", 6: "last", 7: "commit", 8: "publish",
             10: "pass0", 11: "tiles1/met(b0)", 12: "lastwarp/blk", 13: "committed"}
    line = " ".join("%s=%.1f" % (names[i], med([t[i] for t in tr])) for i in sorted(names) if all(t[i] is not None and abs(t[i]) < 1e6 for t in tr))
    print("%s path=%d cold=%d hostlog=%d: events %.1f us (min %.1f)  device %.1f us | %s" % (name, path, cold, host_log, med(ev), min(ev), med(dv), line), flush=True)
    ctx.shutdown()

for name in ("c1", "c3"):
    for path in (cc.CC_PATH_PHASES, cc.CC_PATH_SINGLE_PASS, cc.CC_PATH_SMALL):
        for cold in (1, 0):
            run(name, path, cold)
    for path in (cc.CC_PATH_PHASES, cc.CC_PATH_SINGLE_PASS, cc.CC_PATH_SMALL):
        run(name, path, 1, host_log=True)
