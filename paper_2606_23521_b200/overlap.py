"""Checkpointing next to compute (Fig. 7b "Throughput impact with overlapped delta checkpointing";
L427 "The persistent kernel occupies 1 block out of 188 SMs = 0.53% of GPU resources"):

    python -m paper_2606_23521_b200.overlap [--region-mib 256] [--blocks 1,2,4,8,16,32,64]

For each worker footprint B (persistent CTAs = SMs reserved, out of 148) it measures, with the worker resident:
  copy_alone_GBps   a bandwidth-bound application kernel (torch device-to-device copy of 4 GiB, read+write bytes)
                    while the worker idles                              -> cost of the reserved SMs
  ckpt_alone_ms     device time of one delta-checkpoint task (256 MiB region, 1 % dirty 4 KiB pages, device log)
  copy_with_ckpt_GBps / ckpt_with_copy_ms   both at the same time       -> interference
and, for reference, the copy with no worker at all.  Second part: many small regions at one boundary --
cc_checkpoint_all (4 launches) against a loop of cc_checkpoint_delta (3 launches per region).
Prints one JSON object.
"""
import argparse
import json
import math
import statistics
import time

import torch

from . import binding as cc


def _copy_gbps(dst, src, stream, reps=6):
    torch.cuda.current_stream().synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(reps):
        dst.copy_(src)
    e1.record(stream)
    e1.synchronize()
    return 2 * src.numel() * reps / (e0.elapsed_time(e1) * 1e-3) / 1e9


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--region-mib", type=int, default=256)
    ap.add_argument("--page", type=int, default=4096)
    ap.add_argument("--dirty", type=float, default=0.01)
    ap.add_argument("--blocks", default="1,2,4,8,16,32,64")
    ap.add_argument("--small-regions", type=int, default=48)
    a = ap.parse_args()
    dev = torch.device("cuda", 0)
    P, N = a.page, a.region_mib << 20
    n_pages = N // P
    n_mut = math.ceil(a.dirty * n_pages)
    A = 2 * ((1006 * 7919 + 12345) % 100000) + 1
    g = torch.Generator(device="cuda")
    g.manual_seed(1006)
    cur = torch.randint(0, 256, (N,), dtype=torch.uint8, device=dev, generator=g)
    src = torch.empty(4 << 30, dtype=torch.uint8, device=dev)
    dst = torch.empty_like(src)
    stream = torch.cuda.current_stream()
    per = n_mut * (16 + P) + 32
    out = {"config": {"region_MiB": a.region_mib, "page_bytes": P, "dirty_pages_per_task": n_mut, "sm_count": 148,
                      "copy": "torch copy_ of 4 GiB device to device, GB/s counts read + write"},
           "copy_no_worker_GBps": round(_copy_gbps(dst, src, stream), 1), "footprints": []}
    for B in [int(x) for x in a.blocks.split(",")]:
        ctx = cc.Context(0, ring_capacity=256, worker_blocks=B, max_lifetime_ns=int(120e9))
        ctx.register_region(1, cur, P)
        log = torch.empty(64 * per, dtype=torch.uint8, device=dev)
        ctx.log_attach(log)
        stream.synchronize()
        ctx.worker_start()
        row = {"worker_blocks": B, "sm_share_pct": round(100.0 * B / 148, 2)}
        try:
            row["copy_alone_GBps"] = round(_copy_gbps(dst, src, stream), 1)

            def tasks(n):
                seqs = []
                for t in range(n):
                    hh = (1006 * 2654435761 + t * 40503) & 0xFFFFFFFF
                    ctx.submit(cc.CC_TASK_TEST_MUTATE, region_id=1, arg0=n_mut, arg1=A, arg2=hh)
                    seqs.append(ctx.submit(cc.CC_TASK_DELTA_CKPT, region_id=1, epoch=t))
                return seqs

            def collect(seqs):
                rs = [ctx.wait(s, 60.0) for s in seqs]
                assert all(r.status == 0 and r.n_dirty == n_mut for r in rs)
                ctx.wait(ctx.submit(cc.CC_TASK_LOG_RESET), 60.0)
                return statistics.median([(r.t_end_ns - r.t_start_ns) / 1e6 for r in rs])

            collect(tasks(4))                                        # warm-up
            row["ckpt_alone_ms"] = round(collect(tasks(16)), 4)
            # both: size the task batch to outlast the copies
            n_tasks = min(60, max(8, int(6 * 2 * src.numel() / 6.0e12 * 1e3 / max(row["ckpt_alone_ms"], 1e-3)) + 4))
            seqs = tasks(n_tasks)
            row["copy_with_ckpt_GBps"] = round(_copy_gbps(dst, src, stream), 1)
            row["ckpt_with_copy_ms"] = round(collect(seqs), 4)
            row["tasks_in_flight_during_copy"] = n_tasks
        finally:
            ctx.worker_stop()
        ctx.shutdown()
        out["footprints"].append(row)

    # ---- many small regions at one boundary: batched vs per-region launches ----
    R = a.small_regions
    small_bytes, sp = 4 << 20, 65536                                 # e.g. per-layer adapter shards of 4 MiB, 64 KiB pages
    regs = [torch.randint(0, 256, (small_bytes,), dtype=torch.uint8, device=dev, generator=g) for _ in range(R)]
    ctx = cc.Context(0)
    for i, t in enumerate(regs):
        ctx.register_region(i + 1, t, sp)
    log = torch.empty(R * (small_bytes + 4096), dtype=torch.uint8, device=dev)
    ctx.log_attach(log)
    res = cc.Result()

    def dirty_all():
        for t in regs:
            t[::sp * 8] ^= 1                                          # 1 page in 8 of every region

    def timed(fn, reps=10):
        ts = []
        for _ in range(reps + 2):
            dirty_all()
            ctx.log_reset()
            torch.cuda.synchronize()
            t0 = time.perf_counter_ns()
            fn()
            torch.cuda.synchronize()
            ts.append((time.perf_counter_ns() - t0) / 1e3)
        return statistics.median(ts[2:])

    t_batch = timed(lambda: ctx.checkpoint_all(1, res))
    rb = res.read()

    def loop():
        for i in range(R):
            ctx.checkpoint_delta(i + 1, 1, res)
    t_loop = timed(loop)
    out["many_small_regions"] = {"regions": R, "region_MiB": small_bytes >> 20, "page_bytes": sp,
                                 "dirty_pages_total": int(rb.n_dirty),
                                 "cc_checkpoint_all_us": round(t_batch, 1), "launches_batched": 4,
                                 "loop_of_cc_checkpoint_delta_us": round(t_loop, 1), "launches_loop": 3 * R,
                                 "speedup": round(t_loop / t_batch, 2)}
    ctx.shutdown()
    print(json.dumps(out))


if __name__ == "__main__":
    main()
