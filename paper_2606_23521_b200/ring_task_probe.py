"""Device timeline of ring checkpoint tasks (c5b shape) per task flavour, trace build."""
import ctypes, statistics, sys, os
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import torch
import synth
import paper_2606_23521_b200 as cc
dev = torch.device("cuda:0")
P, n_pages, n_mut = 4096, 65536, 656
N = P * n_pages
A = 2 * ((1006 * 7919 + 12345) % 100000) + 1

def run(flags, host_log, blocks, n=40):
    cur = synth.raw_region(N, 1006, dev)
    ctx = cc.Context(0, ring_capacity=256, worker_blocks=blocks, max_lifetime_ns=int(60e9))
    ctx.register_region(1, cur, P)
    cap = 1 << 30
    log = torch.zeros(cap, dtype=torch.uint8, pin_memory=True) if host_log else torch.zeros(cap, dtype=torch.uint8, device=dev)
    ctx.log_attach(log)
    tbuf = (ctypes.c_uint64 * 32)()
    torch.cuda.synchronize()
    ctx.worker_start()
    devs, trs = [], []
    try:
        ctx.wait(ctx.submit(cc.CC_TASK_LOG_RESET), 30.0)
        for t in range(n):
            ctx.wait(ctx.submit(cc.CC_TASK_TEST_MUTATE, region_id=1, arg0=n_mut, arg1=A, arg2=t), 30.0)
            r = ctx.wait(ctx.submit(cc.CC_TASK_DELTA_CKPT, region_id=1, epoch=t, flags=flags), 30.0)
            assert r.status == 0 and r.n_dirty == n_mut, (r.status, r.n_dirty)
            ctx.wait(ctx.submit(cc.CC_TASK_LOG_RESET), 30.0)
            if t >= 5:
                devs.append((r.t_end_ns - r.t_start_ns) / 1e3)
    finally:
        ctx.worker_stop()
    ctx.lib.cc_debug_trace(ctx.h, tbuf)
    fp = ctx.worker_footprint()
    # trace slots of the LAST task relative to its t_start
    t0 = r.t_start_ns
    tr = {i: (int(tbuf[i]) - t0) / 1e3 for i in (10, 11, 12, 13) if tbuf[i]}
    print("flags=%d hostlog=%d blocks=%d x %d: device p50 %.1f us min %.1f | last task: %s (t_end %.1f)" % (
        flags, host_log, fp["blocks"], fp["threads_per_block"], statistics.median(devs), min(devs),
        " ".join("%d=%.1f" % kv for kv in sorted(tr.items())), (r.t_end_ns - t0) / 1e3), flush=True)
    ctx.shutdown()

for host_log in (0, 1):
    for flags in (0, cc.CC_TASKF_FUSED):
        run(flags, host_log, cc.CC_WORKER_BLOCKS_ALL)
