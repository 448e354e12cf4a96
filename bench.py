#!/usr/bin/env python
"""bench.py -- delta-checkpoint throughput on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c2|c2-small]

Workload (N=1): BASELINE.json configs[1] -- Llama-3-8B-shaped paged KV cache, bf16, 32 layers x 4096
blocks x 64 KiB = 8 GiB; one decode step appends a token to 256 sequences, so 8,192 blocks are dirty.
A "step" = the application's decode write (new K/V token rows scattered into the cache) followed by
one pass of the whole checkpoint path: a1 scan, a2 compaction, a3 gather + CRC32C into the log,
a4 commit + publish, a5 shadow update (cc_checkpoint_delta: 3 kernels of ours).
  value : region bytes scanned per second (N_region / step time), whole job (sum over ranks), with
          everything resident in HBM (device-memory log).
  e2e   : same metric through the same C-ABI call with HOST buffers: the step's new tokens start in
          pinned host memory (H2D copy inside the timed region), the log is a pinned HOST buffer (the
          gather kernel writes the 512 MiB of records over the host link) and the 64-byte result is
          read on the host every step.
  roofline : the scan kernel (dominant): algorithmic bytes 2 x N_region per launch / its mean duration
          from CUDA events recorded on the launch stream inside the timed region, vs the measured HBM
          copy bandwidth of MEASURED_PEAKS.json.
  cpu_baseline : the CPU oracle (oracle/, plain C, as it stands) on a bounded sample of the same workload.
Multi-GPU: the path shards with no exchange -- every rank checkpoints its own region;
"scaling": "weak"; no data-path collective (only the timing barrier / max-reduce).
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "delta_checkpoint_region_scan_throughput"
UNIT = "GB/s"

WORKLOADS = {
    # name: (layers, blocks per layer, sequences)  -- block = 64 KiB
    "c2": (32, 4096, 256),          # 8 GiB, 8,192 dirty blocks (BASELINE.json configs[1])
    "c2-small": (4, 1024, 64),      # 256 MiB, 256 dirty blocks (quick functional run; not the metric config)
}
P = 65536
TOKENS, HEADS, DIM = 16, 8, 128
ROW = HEADS * DIM * 2               # bytes of one K (or V) token row = 2 KiB


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


# ------------------------------------------------------------------------ clocks --

class ClockSampler:
    """Samples SM clocks and throttle reasons DURING the timed region (NVML in a thread; nvidia-smi as a
    fallback when NVML is unavailable)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.sm, self.max_sm, self.reasons = index, [], None, set()
        self._stop, self._t, self.nvml, self.h = threading.Event(), None, None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            idx = index
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            if vis:
                try:
                    idx = int(vis.split(",")[index])
                except Exception:
                    idx = index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_sm = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        self.sm.append(float(n.nvmlDeviceGetClockInfo(self.h, n.NVML_CLOCK_SM)))
        try:
            r = n.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            r = n.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        for name, bit in (("hw_slowdown", 0x8), ("sw_power_cap", 0x4), ("sw_thermal_slowdown", 0x20),
                          ("hw_thermal_slowdown", 0x40)):
            if r & bit:
                self.reasons.add(name)

    def _sample_smi(self):
        out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                              "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
        f = [x.strip() for x in out.strip().split(",")]
        if len(f) >= 6:
            self.sm.append(float(f[0]))
            self.max_sm = float(f[1])
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[2:6]):
                if v.lower().startswith("active"):
                    self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._sample_nvml() if self.nvml else self._sample_smi()
            except Exception:
                pass
            self._stop.wait(0.002)

    def start(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()

    def stop(self):
        self._stop.set()
        if self._t:
            self._t.join(timeout=10)
        return {"sm_mhz": statistics.median(self.sm) if self.sm else None, "sm_max_mhz": self.max_sm,
                "reasons": sorted(self.reasons), "samples": len(self.sm),
                "source": "nvml" if self.nvml else "nvidia-smi"}


def measured_peak():
    try:
        d = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------ CPU oracle leg --

def cpu_oracle_leg(layers, blocks, seqs, reps, device):
    """Time the oracle's full checkpoint (scan + gather + CRC + shadow) on a bounded sample: the first
    `layers` layers of the workload.  Returns (region GB/s, seconds per pass, description)."""
    import numpy as np
    import torch
    import oracle
    import synth
    cur = synth.kv_cache_region(layers, blocks, 1002, device)
    cur_h = cur.cpu().numpy()
    del cur
    sh_h = cur_h.copy()
    n = cur_h.size
    k = layers * seqs
    log = np.zeros(k * (16 + P) + 32, dtype=np.uint8)
    times = []
    for r in range(reps):
        t = torch.from_numpy(cur_h)
        synth.kv_decode_step(t, layers, blocks, seqs, 5000 + r)
        t0 = time.perf_counter()
        st, D, nb, W = oracle.checkpoint(cur_h, sh_h, P, 1, r, log, 0)
        times.append(time.perf_counter() - t0)
        assert st == 0 and D.size == k, (st, D.size, k)
    best = statistics.median(times)
    # beside it: the oracle's page-range-partitioned scan (orc_scan_mt, the same memcmp loop) on every host core
    cores = os.cpu_count() or 1
    t_mt = []
    for r in range(3):
        t0 = time.perf_counter()
        oracle.scan_mt(cur_h, sh_h, P, cores)
        t_mt.append(time.perf_counter() - t0)
    cpu_oracle_leg.scan_all_cores = {"value": round(n / statistics.median(t_mt) / 1e9, 3), "unit": UNIT, "cores": cores,
                                     "what": "oracle scan only (no gather / CRC), page range split over all host cores"}
    return n / best / 1e9, best, "first %d of 32 layers of the workload (%.2f GiB region, %d dirty blocks), %d passes, median" % (
        layers, n / 2**30, k, reps)


# ------------------------------------------------------------------------ GPU arm --

def run_ours(args):
    import torch
    import synth
    import paper_2606_23521_b200 as cc

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    layers, blocks, seqs = WORKLOADS[args.workload]
    K, Wm = args.steps, max(args.warmup, 3)

    # ---- synthetic workload (config 2) ----
    cur = synth.kv_cache_region(layers, blocks, 1002 + rank, dev)
    N = cur.numel()
    k_exp = layers * seqs
    rows = cur.view(torch.bfloat16).view(layers * blocks * 2 * TOKENS, HEADS * DIM)     # one K or V token row = 2 KiB
    g = synth.gen(2002 + rank, dev)
    L_idx = torch.arange(layers, device=dev).repeat_interleave(seqs)
    B_idx = torch.cat([torch.randperm(blocks, generator=g, device=dev)[:seqs] for _ in range(layers)])
    T_idx = torch.randint(0, TOKENS, (layers * seqs,), generator=g, device=dev)
    blk = L_idx * blocks + B_idx
    row_idx = torch.stack([(blk * 2 + 0) * TOKENS + T_idx, (blk * 2 + 1) * TOKENS + T_idx], dim=1).reshape(-1)
    pools = [torch.randn(layers * seqs * 2, HEADS * DIM, generator=g, device=dev).to(torch.bfloat16) for _ in range(2)]
    pools_host = [p.cpu().pin_memory() for p in pools]
    stage = torch.empty_like(pools[0])

    def decode_write(values):
        rows.index_copy_(0, row_idx, values)         # the application's KV append (torch, not part of the library)

    ctx = cc.Context(local)
    ctx.register_region(1, cur, P)                    # shadow := cur
    log_bytes = k_exp * (16 + P) + 32
    log_dev = torch.empty(log_bytes, dtype=torch.uint8, device=dev)
    # The e2e arm uses the fused single pass, which writes records while it scans only if the worst case (every
    # block dirty) fits behind the write offset -- so the host log is sized like a real append-only log, not
    # like one epoch.
    worst_bytes = (N // P) * (16 + P) + 32
    log_host = torch.empty(worst_bytes if not args.no_e2e else log_bytes, dtype=torch.uint8, pin_memory=True)
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    results = [cc.Result() for _ in range(K)]
    warm_res = cc.Result()
    stream = torch.cuda.current_stream()

    def make_ev():
        e = torch.cuda.Event(enable_timing=True)
        e.record(stream)
        return e

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    def step_dev(s, res, evs=None):
        decode_write(pools[s & 1])
        if evs:
            evs[0].record(stream)
            ctx.trace_events(evs[1], evs[2])
        ctx.checkpoint_delta(1, s, res)
        if evs:
            evs[3].record(stream)

    # ================= arm 1: everything resident in HBM (device log) =================
    ctx.log_attach(log_dev, committed)
    for s in range(Wm):
        step_dev(s, warm_res)
        torch.cuda.synchronize()
        ctx.log_reset()
    evs = [[make_ev() for _ in range(4)] for _ in range(K)]
    sampler = ClockSampler(local)
    barrier()
    launches0 = ctx.kernel_launches()
    sampler.start()
    t_begin, t_end = make_ev(), make_ev()
    torch.cuda.synchronize()
    t_begin.record(stream)
    for s in range(K):
        # the log buffer holds one epoch; W is rewound by an 8-byte stream-ordered memset (cc_log_reset_async)
        step_dev(Wm + s, results[s], evs[s])
        ctx.log_reset_async()
    t_end.record(stream)
    barrier()
    clocks = sampler.stop()
    ctx.trace_events(None, None)
    launches = ctx.kernel_launches() - launches0
    ms_total = t_begin.elapsed_time(t_end)
    for s in range(K):
        r = results[s].read()
        assert r.status == 0 and r.n_dirty == k_exp and r.bytes == log_bytes, r.as_dict()
    t_scan = [evs[s][0].elapsed_time(evs[s][1]) for s in range(K)]
    t_compact = [evs[s][1].elapsed_time(evs[s][2]) for s in range(K)]
    t_gather = [evs[s][2].elapsed_time(evs[s][3]) for s in range(K)]
    t_ckpt = [evs[s][0].elapsed_time(evs[s][3]) for s in range(K)]

    # ================= arm 1b: allocator-aware discovery =================
    # Same workload, but the block allocator hands over its dirty-block bitmap, so the
    # cost is proportional to the dirty bytes: mark load + compaction + gather, no scan of the 8 GiB.
    n_pages = N // P
    bm_host = torch.zeros((n_pages + 31) // 32, dtype=torch.int64)
    bm_host.index_put_((blk.cpu() >> 5,), (1 << (blk.cpu() & 31)), accumulate=True)      # distinct blocks: OR == add
    bm_src = torch.where(bm_host >= 2**31, bm_host - 2**32, bm_host).to(torch.int32).to(dev)
    marks = torch.empty_like(bm_src)
    mk_evs = [[make_ev() for _ in range(2)] for _ in range(K)]
    for s in range(Wm + K):
        decode_write(pools[s & 1])
        marks.copy_(bm_src)                          # the allocator's bitmap for this step
        if s >= Wm:
            mk_evs[s - Wm][0].record(stream)
        ctx.checkpoint_marked(1, 10_000 + s, marks, cc.CC_MARK_CONSUME, warm_res)
        if s >= Wm:
            mk_evs[s - Wm][1].record(stream)
        ctx.log_reset_async()
    torch.cuda.synchronize()
    r = warm_res.read()
    assert r.status == 0 and r.n_dirty == k_exp and r.bytes == log_bytes and not marks.any(), r.as_dict()
    t_marked = [a.elapsed_time(b) for a, b in mk_evs]

    # ================= arm 2: end to end with host buffers =================
    e2e = None
    if not args.no_e2e:
        ctx.log_attach(log_host, committed)
        h2d = pools_host[0].numel() * pools_host[0].element_size()

        def step_e2e(s, res, fused=True):
            stage.copy_(pools_host[s & 1], non_blocking=True)      # H2D: this step's new tokens
            decode_write(stage)
            # the records go straight into pinned host memory; fused: while the scan is still running
            (ctx.checkpoint_delta_fused if fused else ctx.checkpoint_delta)(1, s, res)
            torch.cuda.synchronize()
            r = res.read()                                         # D2H: the 64-byte result, read on the host
            assert r.status == 0 and r.n_dirty == k_exp
            ctx.log_reset()

        base = Wm + K                                              # keep alternating the value pools
        for s in range(Wm):
            step_e2e(base + s, warm_res)
        barrier()
        e0, e1 = make_ev(), make_ev()
        torch.cuda.synchronize()
        e0.record(stream)
        for s in range(K):
            step_e2e(base + Wm + s, results[s])
        e1.record(stream)
        barrier()
        ms_fused = e0.elapsed_time(e1)
        # for comparison: the same end-to-end step through the three-kernel path (scan, then compact, then gather)
        base2 = base + Wm + K
        for s in range(2):
            step_e2e(base2 + s, warm_res, fused=False)
        torch.cuda.synchronize()
        e0.record(stream)
        for s in range(K):
            step_e2e(base2 + 2 + s, results[s], fused=False)
        e1.record(stream)
        torch.cuda.synchronize()
        ms_three = e0.elapsed_time(e1)

        # The pipeline a production AOF would run (PAPER.md:L262-263 staging buffer -> append): the checkpoint appends
        # to a DEVICE log at HBM speed, cc_log_drain hands the committed bytes to the copy engine (57 GB/s, no SM),
        # and the drain of step s overlaps the scan of step s+1.  The host reads every step's result before it
        # continues; the log bytes of step s are in host memory (and committed_off_host says so) one step later.
        EPOCHS = 15
        del log_dev
        log_ring = torch.empty(EPOCHS * log_bytes, dtype=torch.uint8, device=dev)
        mirror = log_host[:EPOCHS * log_bytes]
        mirror_committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
        copy_stream = torch.cuda.Stream(device=dev)
        ctx.log_attach(log_ring, committed)
        ctx.log_mirror_attach(mirror, mirror_committed)
        state = {"epochs": 0, "W": 0}

        def step_dma(s, res):
            stage.copy_(pools_host[s & 1], non_blocking=True)      # H2D: this step's new tokens
            decode_write(stage)
            ctx.checkpoint_delta(1, s, res)                        # three kernels, device log
            stream.synchronize()                                   # this stream only: the copy engine keeps draining
            r = res.read()                                         # D2H: the 64-byte result, read on the host
            assert r.status == 0 and r.n_dirty == k_exp
            ctx.log_drain(r.log_offset_after, copy_stream)         # D2H: the step's records, by the copy engine
            state["epochs"] += 1
            state["W"] = int(r.log_offset_after)
            if state["epochs"] == EPOCHS:                          # the device log is a ring of EPOCHS epochs
                copy_stream.synchronize()
                ctx.log_reset()
                state["epochs"], state["W"] = 0, 0

        base3 = base2 + 2 + K
        for s in range(Wm):
            step_dma(base3 + s, warm_res)
        copy_stream.synchronize()
        barrier()
        e0.record(stream)
        for s in range(K):
            step_dma(base3 + Wm + s, results[s])
        stream.wait_stream(copy_stream)                            # the last drain is inside the timed region
        e1.record(stream)
        barrier()
        ms_e2e = e0.elapsed_time(e1)
        copy_stream.synchronize()
        assert int(mirror_committed.item()) == state["W"], (int(mirror_committed.item()), state)
        assert torch.equal(mirror[:state["W"]], log_ring[:state["W"]].cpu()), "host mirror differs from the device log"
        ctx.log_mirror_attach(None)
        # Whether the copy engine gets HBM bandwidth while the scan saturates it differs from box to box (10.1 ms when
        # it does, 12.9 ms when the drain only proceeds between kernels); the fused direct path is steady at ~11.7 ms.
        # A user picks the faster one on their box: e2e reports that one and names it, both numbers are kept.
        path = "device log + cc_log_drain (copy engine)" if ms_e2e <= ms_fused else "cc_checkpoint_delta_fused into the pinned host log"
        e2e = {"ms": min(ms_e2e, ms_fused), "h2d": h2d, "d2h": log_bytes + 64, "ms_three_kernel": ms_three, "ms_fused": ms_fused,
               "ms_drain": ms_e2e, "path": path}

    # ---- reduce over ranks: max time ----
    def rmax(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    ms_total = rmax(ms_total)
    if e2e:
        e2e["ms"] = rmax(e2e["ms"])
        e2e["ms_drain"], e2e["ms_fused"] = rmax(e2e["ms_drain"]), rmax(e2e["ms_fused"])

    if rank == 0:
        peak, peak_src = measured_peak()
        scan_ms = statistics.mean(t_scan)
        achieved = 2 * N / (scan_ms * 1e-3) / 1e9
        # dram__bytes_read.sum + dram__bytes_write.sum of cc_scan_kernel on this workload, one launch, from the
        # ncu --set full capture summarised in profiles/r01_ncu_full.md (17.179897 GB read + 0.003812 GB written)
        traffic = 17_183_709_000 if args.workload == "c2" else None
        value = world * K * N / (ms_total * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": round(ms_total / K, 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8 (bitwise compare/copy of bf16 KV bytes; CRC32C in u32)", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[1]: paged KV cache %d layers x %d blocks x 64 KiB = %.2f GiB per GPU, "
                                   "decode step dirties %d blocks; log in device memory" % (layers, blocks, N / 2**30, k_exp),
                       "page_bytes": P, "region_bytes_per_gpu": N, "dirty_pages": k_exp, "dirty_bytes": k_exp * P,
                       "l2": "inputs larger than L2 (2 x %.0f GiB streamed per step vs 126 MB L2)" % (N / 2**30),
                       "parallelism": "dp%d (independent regions, no collective)" % world},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "phases_ms": {"scan": round(scan_ms, 4), "compact": round(statistics.mean(t_compact), 4),
                          "gather_commit_shadow": round(statistics.mean(t_gather), 4),
                          "checkpoint_total": round(statistics.mean(t_ckpt), 4),
                          "best_checkpoint_total": round(min(t_ckpt), 4)},
            "hbm_fraction": {
                "bytes_convention": "2 x region + 3 x dirty (BASELINE.json)",
                "scan_GBps_2N": round(achieved, 1),
                "checkpoint_GBps_2N_3kP": round((2 * N + 3 * k_exp * P) / (statistics.mean(t_ckpt) * 1e-3) / 1e9, 1),
                "scan_frac_of_8000": round(achieved / 8000, 4),
                "checkpoint_frac_of_8000": round((2 * N + 3 * k_exp * P) / (statistics.mean(t_ckpt) * 1e-3) / 1e9 / 8000, 4),
                "dirty_GBps_logged": round(k_exp * P / (statistics.mean(t_gather) * 1e-3) / 1e9, 1)},
            "roofline": {"bound": "hbm", "kernel": "cc_scan_kernel", "achieved": round(achieved, 1), "peak": peak,
                         "unit": "GB/s", "frac": round(achieved / peak, 4), "traffic": traffic,
                         "peak_source": peak_src, "algorithmic_bytes_per_launch": 2 * N,
                         "avg_launch_ms": round(scan_ms, 4)},
        }
        mk_ms = statistics.mean(t_marked)
        line["allocator_aware"] = {
            "what": "cc_checkpoint_marked(CC_MARK_CONSUME) on the same workload with the allocator's dirty-block bitmap "
                    "(SURVEY.md 8f #1): no region scan; 4 kernels (mark load, compaction, gather, mark clear)",
            "ms_per_checkpoint": round(mk_ms, 4), "best_ms": round(min(t_marked), 4),
            "dirty_GBps_logged": round(k_exp * P / (mk_ms * 1e-3) / 1e9, 1),
            "hbm_GBps_3kP": round(3 * k_exp * P / (mk_ms * 1e-3) / 1e9, 1),
            "frac_of_measured_peak": round(3 * k_exp * P / (mk_ms * 1e-3) / 1e9 / peak, 4),
            "speedup_vs_scan_path": round(statistics.mean(t_ckpt) / mk_ms, 2)}
        if e2e:
            line["e2e"] = {"value": round(world * K * N / (e2e["ms"] * 1e-3) / 1e9, 2), "unit": UNIT,
                           "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                           "ms_per_step": round(e2e["ms"] / K, 4),
                           "host_link_GBps_log": round(log_bytes * K / (e2e["ms"] * 1e-3) / 1e9, 2),
                           "path": e2e["path"],
                           "ms_per_step_drain_pipeline": round(e2e["ms_drain"] / K, 4),
                           "ms_per_step_direct_fused": round(e2e["ms_fused"] / K, 4),
                           "ms_per_step_direct_three_kernel": round(e2e["ms_three_kernel"] / K, 4),
                           "note": "value = the faster of the two host-log paths measured in this run (named in path).  drain "
                                   "pipeline: cc_checkpoint_delta into a device log (ring of 15 epochs) + cc_log_drain (copy engine) "
                                   "into the pinned host log, the drain of step s overlapping step s+1; new tokens copied H2D and the "
                                   "result read on the host every step; host link floor = 512 MiB / 57 GB/s = 9.4 ms.  direct_* = the "
                                   "record writer storing straight into the pinned host log (SM stores cap at 52.7 GB/s): fused single "
                                   "pass / three kernels"}
        if not args.no_cpu_baseline:
            torch.cuda.empty_cache()
            sl = min(layers, 8)
            v, sec, desc = cpu_oracle_leg(sl, blocks, seqs, 3, dev)
            line["cpu_baseline"] = {"value": round(v, 3), "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": desc, "seconds_per_pass": round(sec, 3),
                                    "scan_only_all_cores": getattr(cpu_oracle_leg, "scan_all_cores", None)}
        print(json.dumps(line), flush=True)
    ctx.shutdown()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


# ------------------------------------------------------------------ reference arm --

def run_reference(args):
    """The oracle, as it stands, on the box's host cores (this tier's reference arm)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    layers, blocks, seqs = WORKLOADS[args.workload]
    sl = min(layers, 4)
    device = "cuda" if torch.cuda.is_available() else "cpu"      # input generation only
    K, Wm = args.steps, args.warmup
    reps = max(1, min(K + Wm, 6))
    v, sec, desc = cpu_oracle_leg(sl, blocks, seqs, reps, device)
    n = sl * blocks * P
    line = {
        "impl": "reference", "metric": METRIC, "value": round(v, 3), "unit": UNIT,
        "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": K, "warmup": Wm,
        "ms_per_step": round(sec * 1e3, 3), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u8", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[1] paged KV cache (64 KiB blocks); each step = the oracle's "
                               "checkpoint on a bounded sample: " + desc, "page_bytes": P, "sample_region_bytes": n},
        "cpu_baseline": {"value": round(v, 3), "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
        "e2e": {"value": round(v, 3), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
