#!/usr/bin/env python
"""bench.py -- delta-checkpoint throughput on B200 (BASELINE.json metric), one JSON line per run.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload c2|c1|c3|c4-sparse|c4-full|c5a|c5b|c2-small]

Default workload (the metric configuration, BASELINE.json configs[1]) = c2: Llama-3-8B-shaped paged KV cache, bf16,
32 layers x 4096 blocks x 64 KiB = 8 GiB; one decode step appends a token to 256 sequences, so 8,192 blocks are dirty.
A "step" = the application's decode write followed by one pass of the whole checkpoint path (a1 scan, a2 compaction,
a3 gather + CRC32C into the log, a4 commit + publish, a5 shadow update) through the C-ABI call cc_checkpoint_delta.
The other workloads are BASELINE.json's remaining configurations; every workload prints the
same JSON shape and checks its result against the CPU oracle in an UNTIMED leg of the same process ("parity"):
  c1        64 MiB raw bytes, 4 KiB pages, 1 % dirty (164 pages), checkpoint + apply round trip
  c3        LoRA adapters, 64 MiB, 64 KiB pages, 5 % dirty (52 pages), bitwise fp32 deltas
  c4-sparse 64 GiB bf16 region, 0.1 % of the pages dirty, page size swept over 4 / 16 / 64 KiB (scan-bound)
  c4-full   100 % dirty (gather/log-bound): 32 GiB with a device log at 4 / 16 / 64 KiB (the largest slice whose log
            fits beside region and shadow, SURVEY.md 8d fallback ii) and, as e2e, the 64 GiB arena as 8 x 8 GiB
            regions drained through one pinned 8.1 GiB host log (fallback i)
  c5a       recovery: replay of a 10,000-record committed log (mixed 4-64 KiB pages) into an 8 GiB arena
  c5b       10,000 checkpoint tasks through the ring buffer / persistent worker on a 256 MiB region at 1 % dirty
  overlap   (not a BASELINE config; Fig. 7b / L427) a bandwidth-bound copy next to the persistent worker at several
            worker footprints, and many small regions at one boundary (cc_checkpoint_all vs a loop)
Keys:
  value    whole-job throughput with inputs resident in HBM when the timed region starts (device-memory log)
  e2e      the same metric through the same C-ABI with HOST buffers (pinned host log or host mirror, inputs copied
           H2D and the 64-byte result read on the host inside the timed region)
  roofline the workload's dominant kernel: algorithmic bytes per launch / its mean duration from CUDA events recorded
           on the launch stream inside the timed region, vs MEASURED_PEAKS.json's HBM copy bandwidth
  cpu_baseline  the CPU oracle (oracle/, plain C, as it stands) on a bounded sample of the same workload
Multi-GPU: the path shards with no exchange -- every rank checkpoints its own region; "scaling":
"weak"; no data-path collective (only the timing barrier / max-reduce).
"""
import argparse
import csv
import json
import math
import os
import statistics
import struct
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "delta_checkpoint_region_scan_throughput"
UNIT = "GB/s"
METRICS = {"c5a": "recovery_log_replay_throughput", "c5b": "ring_checkpoint_task_throughput",
           "overlap": "copy_throughput_next_to_checkpoint_worker"}
KV = {"c2": (32, 4096, 256), "c2-small": (4, 1024, 64)}       # layers, blocks per layer, sequences; block = 64 KiB
P_KV = 65536
TOKENS, HEADS, DIM = 16, 8, 128
WORKLOADS = ["c1", "c2", "c2-small", "c3", "c4-sparse", "c4-full", "c5a", "c5b", "overlap"]


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=WORKLOADS)
    ap.add_argument("--large-gib", type=int, default=64, help="c4: region size (halved until it fits)")
    ap.add_argument("--tasks", type=int, default=10000, help="c5b: ring tasks")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-parity", action="store_true", help="skip the untimed oracle comparison (profiling runs)")
    ap.add_argument("--no-extras", action="store_true", help="c2: skip the allocator-aware and ring legs")
    ap.add_argument("--no-configs", action="store_true", help="c2: skip the short legs of the other configs (c1, c3, c5a, c5b)")
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
        return self

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


def ncu_traffic(kernel, workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel`, read at run time from the newest tracked
    `ncu --set full` summary of this workload (profiles/rNN_ncu_full[_<workload>].csv).  `kernel` may be a tuple of names or
    name prefixes ending in '*': then the sum over the FIRST launch of every kernel that matches (a call that is several
    launches; a capture file holds one call).  Returns (bytes or None, source)."""
    if isinstance(kernel, (tuple, list)):
        return _ncu_traffic_sum(tuple(kernel), workload)
    pdir = os.path.join(ROOT, "profiles")
    suffix = "" if workload == "c2" else "_" + workload.replace("-", "_")
    try:
        names = sorted(f for f in os.listdir(pdir) if f.endswith("_ncu_full%s.csv" % suffix) and f[0] == "r" and f[1:3].isdigit())
    except OSError:
        names = []
    for name in reversed(names):
        try:
            with open(os.path.join(pdir, name), newline="") as fh:
                for row in csv.DictReader(fh):
                    if row.get("Kernel Name", "").split("(")[0].strip() == kernel:
                        tot = 0.0
                        for col, val in row.items():                       # ncu picks the unit per column
                            if col.startswith("dram__bytes_read.sum") or col.startswith("dram__bytes_write.sum"):
                                unit = col[col.index("[") + 1:col.index("]")].lower()
                                tot += float(val) * {"byte": 1.0, "kbyte": 1e3, "mbyte": 1e6, "gbyte": 1e9, "tbyte": 1e12}[unit]
                        return int(round(tot)), "profiles/%s (one ncu --set full launch of %s)" % (name, kernel)
        except Exception:
            continue
    return None, "no tracked ncu --set full capture of %s on this workload" % kernel


def _ncu_traffic_sum(patterns, workload):
    pdir = os.path.join(ROOT, "profiles")
    suffix = "" if workload == "c2" else "_" + workload.replace("-", "_")
    try:
        names = sorted(f for f in os.listdir(pdir) if f.endswith("_ncu_full%s.csv" % suffix) and f[0] == "r" and f[1:3].isdigit())
    except OSError:
        names = []
    hit = lambda k: any(k == p or (p.endswith("*") and k.startswith(p[:-1])) for p in patterns)
    for name in reversed(names):
        try:
            seen, tot = [], 0.0
            with open(os.path.join(pdir, name), newline="") as fh:
                for row in csv.DictReader(fh):
                    k = row.get("Kernel Name", "").split("(")[0].strip()
                    if not hit(k) or k in seen:
                        continue
                    seen.append(k)
                    for col, val in row.items():
                        if col.startswith("dram__bytes_read.sum") or col.startswith("dram__bytes_write.sum"):
                            unit = col[col.index("[") + 1:col.index("]")].lower()
                            tot += float(val) * {"byte": 1.0, "kbyte": 1e3, "mbyte": 1e6, "gbyte": 1e9, "tbyte": 1e12}[unit]
            if seen:
                return int(round(tot)), "profiles/%s (ncu --set full, one launch each of %s)" % (name, ", ".join(seen))
        except Exception:
            continue
    return None, "no tracked ncu --set full capture of %s on this workload" % (patterns,)


def roofline(kernel, algo_bytes, ms, workload, kernels=None):
    """kernel: the name reported; kernels: the launches whose DRAM traffic is summed (default: `kernel` itself)."""
    peak, peak_src = measured_peak()
    ach = algo_bytes / (ms * 1e-3) / 1e9
    traffic, tsrc = ncu_traffic(kernels if kernels is not None else kernel, workload)
    return {"bound": "hbm", "kernel": kernel, "achieved": round(ach, 1), "peak": peak, "unit": "GB/s",
            "frac": round(ach / peak, 4), "frac_of_8000": round(ach / 8000, 4), "traffic": traffic, "traffic_source": tsrc,
            "peak_source": peak_src, "algorithmic_bytes_per_launch": int(algo_bytes), "avg_launch_ms": round(ms, 4)}


class Env:
    """torch / rank / stream plumbing shared by the workloads."""

    def __init__(self):
        import torch
        self.torch = torch
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
            self.dist = dist
        torch.cuda.set_device(self.local)
        self.dev = torch.device("cuda", self.local)
        self.stream = torch.cuda.current_stream()
        self._flush = None

    def ev(self):
        e = self.torch.cuda.Event(enable_timing=True)
        e.record(self.stream)
        return e

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.dist is not None:
            self.dist.barrier()
            self.torch.cuda.synchronize()

    def rmax(self, x):
        if self.dist is None:
            return x
        t = self.torch.tensor([x], dtype=self.torch.float64, device=self.dev)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def flush_l2(self, it=0):
        """Write a 512 MiB buffer (> 126 MB L2) so that the next checkpoint starts cold."""
        if self._flush is None:
            self._flush = self.torch.empty(512 << 20, dtype=self.torch.uint8, device=self.dev)
        self._flush.fill_(it & 0xFF)

    def finish(self):
        if self.dist is not None:
            self.dist.barrier()
            self.dist.destroy_process_group()


def emit(args, line):
    """Print the workload's JSON line -- or hand it to the caller that runs this workload as a short leg of another line."""
    sink = getattr(args, "collect", None)
    if sink is not None:
        sink.append(line)
    else:
        print(json.dumps(line), flush=True)


def base_line(env, K, Wm, value, ms_per_step, workload_desc, extra_cfg, dtype):
    cfg = {"workload": workload_desc, "parallelism": "dp%d (independent regions, no collective)" % env.world}
    cfg.update(extra_cfg)
    return {"metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": env.world, "steps": K, "warmup": Wm,
            "ms_per_step": round(ms_per_step, 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": dtype, "data": "synthetic", "config": cfg}


# ------------------------------------------------------------ oracle legs (CPU) --
# One function per workload: times the oracle, as it stands, on a bounded sample.  Used by cpu_baseline (our arm) and by
# --impl reference, so that both report the SAME sample.  Returns dict(value, seconds_per_pass, cores, sample).

def _passes(fn, reps):
    ts = []
    for r in range(reps):
        t0 = time.perf_counter()
        fn(r)
        ts.append(time.perf_counter() - t0)
    return statistics.median(ts)


def oracle_leg_kv(workload, reps=5):
    import numpy as np
    import torch
    import oracle
    import synth
    layers, blocks, seqs = KV[workload]
    sl = min(layers, 8)                                        # first 8 of 32 layers: 2 GiB of the 8 GiB workload
    dev = "cuda" if torch.cuda.is_available() else "cpu"       # input generation only
    cur_h = synth.kv_cache_region(sl, blocks, 1002, dev).cpu().numpy()
    sh_h = cur_h.copy()
    n, k = cur_h.size, sl * seqs
    log = np.zeros(k * (16 + P_KV) + 32, dtype=np.uint8)
    times = []
    for r in range(reps):
        synth.kv_decode_step(torch.from_numpy(cur_h), sl, blocks, seqs, 5000 + r)
        t0 = time.perf_counter()
        st, D, nb, W = oracle.checkpoint(cur_h, sh_h, P_KV, 1, r, log, 0)
        times.append(time.perf_counter() - t0)
        assert st == 0 and D.size == k, (st, D.size, k)
    sec = statistics.median(times)
    cores = os.cpu_count() or 1
    t_mt = _passes(lambda r: oracle.scan_mt(cur_h, sh_h, P_KV, cores), 3)
    return {"value": round(n / sec / 1e9, 3), "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "first %d of %d layers of the workload (%.2f GiB region, %d dirty blocks), %d passes, median; "
                      "the same sample in cpu_baseline and in --impl reference" % (sl, layers, n / 2**30, k, reps),
            "seconds_per_pass": round(sec, 4),
            "scan_only_all_cores": {"value": round(n / t_mt / 1e9, 3), "unit": UNIT, "cores": cores,
                                    "what": "oracle scan only (orc_scan_mt: the same memcmp loop, page range split over all host cores)"}}


def oracle_leg_region(make, P, rearm_host, k_expect, desc, reps=5):
    """Generic: make() -> host numpy region; rearm_host(cur, r) mutates it; times oracle.checkpoint on all of it."""
    import numpy as np
    import oracle
    cur_h = make()
    sh_h = cur_h.copy()
    n = cur_h.size
    n_pages = (n + P - 1) // P
    log = np.zeros(min(n_pages, max(k_expect, 1)) * (16 + P) + 32, dtype=np.uint8)
    times = []
    for r in range(reps):
        rearm_host(cur_h, r)
        t0 = time.perf_counter()
        st, D, nb, W = oracle.checkpoint(cur_h, sh_h, P, 1, r, log, 0)
        times.append(time.perf_counter() - t0)
        assert st == 0 and D.size == k_expect, (st, D.size, k_expect)
    sec = statistics.median(times)
    return {"value": round(n / sec / 1e9, 3), "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "%s, %d passes, median" % (desc, reps), "seconds_per_pass": round(sec, 4)}


def _np_toggle(cur_h, offs, masks):
    cur_h[offs] ^= masks


def oracle_leg(workload, args):
    import numpy as np
    import torch
    import synth
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    if workload in KV:
        return oracle_leg_kv(workload)
    if workload == "c1":
        cur = synth.raw_region(64 << 20, 1001, dev)
        pages, offs, masks = synth.sparse_xor_flips(cur, 4096, 0.01, 1001)
        synth.toggle_flips(cur, offs, masks)
        o, m = offs.cpu().numpy(), masks.cpu().numpy()
        return oracle_leg_region(lambda: cur.cpu().numpy(), 4096, lambda c, r: _np_toggle(c, o, m), len(pages),
                                 "the whole workload (64 MiB, 164 dirty 4 KiB pages)", reps=9)
    if workload == "c3":
        cur = synth.lora_region(32, 1003, dev)
        host = cur.cpu()

        def rearm(c, r):
            got = synth.lora_update(torch.from_numpy(c), 65536, 0.05, 4000 + r)
            assert len(got) == 52
        return oracle_leg_region(lambda: host.numpy().copy(), 65536, rearm, 52,
                                 "the whole workload (64 MiB, 52 dirty 64 KiB pages)", reps=9)
    if workload in ("c4-sparse", "c4-full"):
        P = 65536
        ratio = 0.001 if workload == "c4-sparse" else 1.0
        N = (2 << 30) if ratio < 1 else (1 << 30)             # first 2 GiB (sparse) / 1 GiB (all dirty: CRC-bound) of the region
        cur = synth.bf16_normal_region(N, 1004, dev)
        pages, offs, masks = synth.sparse_xor_flips(cur, P, ratio, 1004 + P)
        synth.toggle_flips(cur, offs, masks)
        o, m = offs.cpu().numpy(), masks.cpu().numpy()
        return oracle_leg_region(lambda: cur.cpu().numpy(), P, lambda c, r: _np_toggle(c, o, m), len(pages),
                                 "first %d GiB of the region at 64 KiB pages, %s" % (N >> 30, "0.1 % dirty" if ratio < 1 else "all pages dirty"),
                                 reps=5)
    if workload == "c5a":
        import oracle
        arena_bytes = 8 << 30
        olog, W, n_rec, views = build_c5a_log(arena_bytes)
        arena = synth.raw_region(arena_bytes, 1005, dev).cpu().numpy()
        regs = [oracle.Region(rid, P, arena[o:o + sz]) for rid, (o, sz, P) in views.items()]
        sec = _passes(lambda r: oracle.apply_log(olog, W, regs), 5)
        return {"value": round(W / sec / 1e9, 3), "unit": UNIT, "cores": 1, "kind": "oracle",
                "sample": "the whole workload (oracle apply of the %d-byte, %d-record log into the 8 GiB arena), 5 passes, median; "
                          "value = log GB/s" % (W, n_rec), "seconds_per_pass": round(sec, 4)}
    if workload == "c5b":
        P, n_pages, n_mut = 4096, 65536, 656
        cur = synth.raw_region(P * n_pages, 1006, dev)
        A = 2 * ((1006 * 7919 + 12345) % 100000) + 1

        def rearm(c, r):
            pages, h = synth.worker_mutation_pages(r, n_pages, n_mut, 1006)
            for j, p in enumerate(pages):
                c[p * P + (h + j) % P] ^= 0x5A
        return oracle_leg_region(lambda: cur.cpu().numpy(), P, rearm, n_mut,
                                 "one task of the workload per pass (256 MiB region, 656 dirty 4 KiB pages)", reps=9)
    raise ValueError(workload)


def build_c5a_log(arena_bytes):
    """Config 5a's committed log, written by the ORACLE's record writer (never by the CUDA path): 100 epochs x 100
    records, epoch e on region (e mod 3)+1 of the arena split (4 / 16 / 64 KiB pages)."""
    import numpy as np
    import oracle
    import synth
    unit = arena_bytes // 8
    eps = synth.recovery_epochs(arena_bytes, 100, 100, 1005, forced_repeats=50)
    n_rec = sum(e.pages.numel() for e in eps)
    cap = sum(e.payloads.numel() + 16 * e.pages.numel() + 32 for e in eps)
    olog = np.zeros(cap, dtype=np.uint8)
    views = {rid: (o8 * unit, s8 * unit, P) for rid, o8, s8, P in synth.C5A_REGIONS}
    W = 0
    for e in eps:
        o, sz, P = views[e.region_id]
        st, W = oracle.write_epoch(olog, W, e.region_id, e.epoch, sz, P, e.pages.numpy(), e.payloads.numpy())
        assert st == 0
    return olog, W, n_rec, views


# ------------------------------------------------------------------ c2 (default) --

def run_c2(args, env):
    import numpy as np
    import synth
    import paper_2606_23521_b200 as cc
    torch, dev, stream, rank, world = env.torch, env.dev, env.stream, env.rank, env.world
    layers, blocks, seqs = KV[args.workload]
    K, Wm = args.steps, max(args.warmup, 3)
    P = P_KV
    ROW = HEADS * DIM

    # ---- synthetic workload (config 2) ----
    cur = synth.kv_cache_region(layers, blocks, 1002 + rank, dev)
    N = cur.numel()
    k_exp = layers * seqs
    rows = cur.view(torch.bfloat16).view(layers * blocks * 2 * TOKENS, ROW)     # one K or V token row = 2 KiB
    g = synth.gen(2002 + rank, dev)
    L_idx = torch.arange(layers, device=dev).repeat_interleave(seqs)
    B_idx = torch.cat([torch.randperm(blocks, generator=g, device=dev)[:seqs] for _ in range(layers)])
    T_idx = torch.randint(0, TOKENS, (layers * seqs,), generator=g, device=dev)
    blk = L_idx * blocks + B_idx
    row_idx = torch.stack([(blk * 2 + 0) * TOKENS + T_idx, (blk * 2 + 1) * TOKENS + T_idx], dim=1).reshape(-1)
    pools = [torch.randn(layers * seqs * 2, ROW, generator=g, device=dev).to(torch.bfloat16) for _ in range(2)]
    pools_host = [p.cpu().pin_memory() for p in pools]
    stage = torch.empty_like(pools[0])

    wstate = {"n": 0}

    def decode_write(values):
        rows.index_copy_(0, row_idx, values)         # the application's KV append (torch, not part of the library)
        wstate["n"] += 1

    def next_pool():
        return wstate["n"] & 1                       # consecutive writes alternate the two value pools: every step dirties k_exp blocks

    ctx = cc.Context(env.local)
    shadow = ctx.register_region(1, cur, P)          # shadow := cur
    log_bytes = k_exp * (16 + P) + 32
    log_dev = torch.empty(log_bytes, dtype=torch.uint8, device=dev)
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    results = [cc.Result() for _ in range(K)]
    warm_res = cc.Result()

    # ================= parity (untimed): this process's CUDA path against the oracle =================
    parity = None
    if not args.no_parity and rank == 0:
        import oracle
        ctx.log_attach(log_dev, committed)
        host_old = cur.cpu().numpy()                                         # == shadow
        decode_write(pools[next_pool()])
        ctx.checkpoint_delta(1, 4242, warm_res)
        torch.cuda.synchronize()
        r = warm_res.read()
        host_new = cur.cpu().numpy()
        olog = np.zeros(log_bytes, dtype=np.uint8)
        st, D, nb, W = oracle.checkpoint(host_new, host_old, P, 1, 4242, olog, 0)   # host_old becomes the oracle's shadow
        ok = ((r.status, r.n_dirty, r.bytes) == (st, D.size, nb) and ctx.dirty_list(1).tolist() == D.tolist()
              and np.array_equal(log_dev.cpu().numpy(), olog) and torch.equal(shadow, cur))
        assert ok, "CUDA path differs from the oracle on the benchmark workload"
        parity = {"checked": "dirty list, all %d log bytes, shadow: bit-exact with oracle.checkpoint on the full %.0f GiB region"
                             % (nb, N / 2**30), "ok": True}
        del host_old, host_new, olog
        ctx.log_reset()

    def step_dev(s, res, evs=None):
        decode_write(pools[next_pool()])
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
    evs = [[env.ev() for _ in range(4)] for _ in range(K)]
    sampler = ClockSampler(env.local)
    env.barrier()
    launches0 = ctx.kernel_launches()
    sampler.start()
    t_begin, t_end = env.ev(), env.ev()
    torch.cuda.synchronize()
    t_begin.record(stream)
    for s in range(K):
        # the log buffer holds one epoch; W is rewound by a one-thread stream-ordered kernel (cc_log_reset_async)
        step_dev(Wm + s, results[s], evs[s])
        ctx.log_reset_async()
    t_end.record(stream)
    env.barrier()
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
    t_marked = None
    if not args.no_extras:
        n_pages = N // P
        bm_host = torch.zeros((n_pages + 31) // 32, dtype=torch.int64)
        bm_host.index_put_((blk.cpu() >> 5,), (1 << (blk.cpu() & 31)), accumulate=True)      # distinct blocks: OR == add
        bm_src = torch.where(bm_host >= 2**31, bm_host - 2**32, bm_host).to(torch.int32).to(dev)
        marks = torch.empty_like(bm_src)
        mk_evs = [[env.ev() for _ in range(2)] for _ in range(K)]
        for s in range(Wm + K):
            decode_write(pools[next_pool()])
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
    # THE e2e pipeline (PAPER.md:L262-263 staging buffer -> append): the checkpoint appends to a DEVICE log at HBM speed;
    # the library's drainer thread (cc_log_drain_start) hands every committed byte range to the copy engine, which
    # carries it into the pinned HOST log while the next step's scan runs.  Every step copies its new tokens H2D and
    # reads the 64-byte result on the host; the timed region ends when the last byte has landed in host memory.
    e2e = None
    if not args.no_e2e:
        EPOCHS = 15
        h2d = pools_host[0].numel() * pools_host[0].element_size()
        del log_dev
        torch.cuda.empty_cache()
        log_ring = torch.empty(EPOCHS * log_bytes, dtype=torch.uint8, device=dev)
        worst_bytes = (N // P) * (16 + P) + 32
        log_host = torch.empty(max(worst_bytes, EPOCHS * log_bytes), dtype=torch.uint8, pin_memory=True)
        mirror = log_host[:EPOCHS * log_bytes]
        mirror_committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
        ctx.log_attach(log_ring, committed)
        ctx.log_mirror_attach(mirror, mirror_committed)
        ctx.log_drain_start()
        state = {"epochs": 0, "W": 0}

        def step_drain(s, res):
            stage.copy_(pools_host[next_pool()], non_blocking=True)      # H2D: this step's new tokens
            decode_write(stage)
            ctx.checkpoint_delta(1, s, res)                        # device log
            stream.synchronize()                                   # this stream only: the copy engine keeps draining
            r = res.read()                                         # D2H: the 64-byte result, read on the host
            assert r.status == 0 and r.n_dirty == k_exp
            state["epochs"] += 1
            state["W"] = int(r.log_offset_after)
            if state["epochs"] == EPOCHS:                          # the device log is a ring of EPOCHS epochs
                ctx.log_drain_wait(state["W"])
                ctx.log_reset()
                state["epochs"], state["W"] = 0, 0

        base = Wm + K
        for s in range(Wm):
            step_drain(base + s, warm_res)
        ctx.log_drain_wait(state["W"])
        env.barrier()
        e0, e1 = env.ev(), env.ev()
        e0.record(stream)
        for s in range(K):
            step_drain(base + Wm + s, results[s])
        ctx.log_drain_wait(state["W"])                             # the last drain is inside the timed region
        e1.record(stream)
        env.barrier()
        ms_drain = e0.elapsed_time(e1)       # e1 is recorded after the host has seen the last byte land
        assert int(mirror_committed.item()) == state["W"], (int(mirror_committed.item()), state)
        assert torch.equal(mirror[:state["W"]], log_ring[:state["W"]].cpu()), "host mirror differs from the device log"
        ctx.log_drain_stop()
        ctx.log_mirror_attach(None)

        # extras, same host-buffer step with the record writer storing straight into the pinned host log
        ctx.log_attach(log_host, committed)

        def step_direct(s, res, fused):
            stage.copy_(pools_host[next_pool()], non_blocking=True)
            decode_write(stage)
            (ctx.checkpoint_delta_fused if fused else ctx.checkpoint_ex)(1, s, res, **({} if fused else {"path": cc.CC_PATH_PHASES}))
            torch.cuda.synchronize()
            r = res.read()
            assert r.status == 0 and r.n_dirty == k_exp
            ctx.log_reset()

        extras = {}
        base2 = base + Wm + K
        for name, fused in (("direct_fused", True), ("direct_three_kernel", False)):
            for s in range(2):
                step_direct(base2 + s, warm_res, fused)
            torch.cuda.synchronize()
            e0.record(stream)
            for s in range(K):
                step_direct(base2 + 2 + s, results[s], fused)
            e1.record(stream)
            torch.cuda.synchronize()
            extras[name] = e0.elapsed_time(e1)
            base2 += 2 + K
        e2e = {"ms": ms_drain, "h2d": h2d, "d2h": log_bytes + 64, "extras": extras}
        del log_ring, log_host, mirror
        torch.cuda.empty_cache()

    # ================= arm 3: the same checkpoint through the ring / persistent worker =================
    ring = None
    if not args.no_extras and rank == 0:
        ring = ring_on_region(cc, env, cur, shadow, P, k_exp, log_bytes, lambda s: decode_write(pools[next_pool()]))

    ms_total = env.rmax(ms_total)
    if e2e:
        e2e["ms"] = env.rmax(e2e["ms"])

    if rank == 0:
        scan_ms = statistics.mean(t_scan)
        value = world * K * N / (ms_total * 1e-3) / 1e9
        line = base_line(env, K, Wm, value, ms_total / K,
                         "BASELINE.json configs[1]: paged KV cache %d layers x %d blocks x 64 KiB = %.2f GiB per GPU, decode step "
                         "dirties %d blocks; log in device memory" % (layers, blocks, N / 2**30, k_exp),
                         {"page_bytes": P, "region_bytes_per_gpu": N, "dirty_pages": k_exp, "dirty_bytes": k_exp * P,
                          "l2": "inputs larger than L2 (2 x %.0f GiB streamed per step vs 126 MB L2)" % (N / 2**30)},
                         "u8 (bitwise compare/copy of bf16 KV bytes; CRC32C in u32)")
        line["gpu_launches"] = int(launches)
        line["clocks"] = clocks
        line["parity"] = parity
        ck = statistics.mean(t_ckpt)
        line["phases_ms"] = {"scan": round(scan_ms, 4), "compact": round(statistics.mean(t_compact), 4),
                             "gather_commit_shadow": round(statistics.mean(t_gather), 4),
                             "checkpoint_total": round(ck, 4), "best_checkpoint_total": round(min(t_ckpt), 4)}
        line["hbm_fraction"] = {
            "bytes_convention": "2 x region + 3 x dirty (BASELINE.json)",
            "scan_GBps_2N": round(2 * N / (scan_ms * 1e-3) / 1e9, 1),
            "checkpoint_GBps_2N_3kP": round((2 * N + 3 * k_exp * P) / (ck * 1e-3) / 1e9, 1),
            "scan_frac_of_8000": round(2 * N / (scan_ms * 1e-3) / 1e9 / 8000, 4),
            "checkpoint_frac_of_8000": round((2 * N + 3 * k_exp * P) / (ck * 1e-3) / 1e9 / 8000, 4),
            "dirty_GBps_logged": round(k_exp * P / (statistics.mean(t_gather) * 1e-3) / 1e9, 1)}
        line["roofline"] = roofline("cc_scan_kernel", 2 * N, scan_ms, args.workload)
        if t_marked:
            mk_ms = statistics.mean(t_marked)
            peak = line["roofline"]["peak"]
            line["allocator_aware"] = {
                "what": "cc_checkpoint_marked(CC_MARK_CONSUME) on the same workload with the allocator's dirty-block bitmap "
                        "(SURVEY.md 8f #1): no region scan",
                "ms_per_checkpoint": round(mk_ms, 4), "best_ms": round(min(t_marked), 4),
                "dirty_GBps_logged": round(k_exp * P / (mk_ms * 1e-3) / 1e9, 1),
                "hbm_GBps_3kP": round(3 * k_exp * P / (mk_ms * 1e-3) / 1e9, 1),
                "frac_of_measured_peak": round(3 * k_exp * P / (mk_ms * 1e-3) / 1e9 / peak, 4),
                "speedup_vs_scan_path": round(ck / mk_ms, 2)}
        if ring:
            line["ring_worker"] = ring
        if e2e:
            line["e2e"] = {"value": round(world * K * N / (e2e["ms"] * 1e-3) / 1e9, 2), "unit": UNIT,
                           "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                           "ms_per_step": round(e2e["ms"] / K, 4),
                           "host_link_GBps_log": round(log_bytes * K / (e2e["ms"] * 1e-3) / 1e9, 2),
                           "path": "cc_checkpoint_delta into a device log (ring of 15 epochs) + the library's drainer thread "
                                   "(cc_log_drain_start: copy engine -> pinned host log, overlapping the next step's scan); new tokens "
                                   "copied H2D and the result read on the host every step; ends when the last byte is in host memory; "
                                   "host link floor = 512 MiB / 57 GB/s = 9.4 ms",
                           "other_paths_ms_per_step": {k2: round(v / K, 4) for k2, v in e2e["extras"].items()},
                           "other_paths": "the record writer storing straight into the pinned host log (SM stores cap at 52.7 GB/s): "
                                          "fused single pass / three kernels"}
        if args.workload == "c2" and world == 1 and not args.no_extras and not args.no_configs:
            ctx.shutdown()                                           # (idempotent; the legs make their own contexts)
            torch.cuda.empty_cache()
            line["configs"] = short_config_legs(args, env)
        if not args.no_cpu_baseline:
            torch.cuda.empty_cache()
            line["cpu_baseline"] = oracle_leg(args.workload, args)
        print(json.dumps(line), flush=True)
    ctx.shutdown()


def short_config_legs(args, env):
    """BASELINE.json's other single-GPU configs as SHORT legs of the default line, so that the driver's record of
    `python bench.py` carries a number and a parity flag for each (the full lines: --workload c1|c3|c5a|c5b).  Same code
    as those workloads, fewer steps / tasks, no CPU baseline, no end-to-end leg."""
    import argparse
    legs = {}
    for name, fn, over in (("c1", lambda a: small_region_workload(a, env, "c1"), {"steps": 10}),
                           ("c3", lambda a: small_region_workload(a, env, "c3"), {"steps": 10}),
                           ("c5a", lambda a: run_c5a(a, env), {"steps": 5}),
                           ("c5b", lambda a: run_c5b(a, env), {"tasks": 1000})):
        sub = argparse.Namespace(**vars(args))
        sub.workload, sub.warmup, sub.no_cpu_baseline, sub.no_e2e, sub.collect = name, 3, True, True, []
        for k2, v in over.items():
            setattr(sub, k2, v)
        t0 = time.perf_counter()
        try:
            fn(sub)
            ln = sub.collect[0]
            rf = ln.get("roofline", {})
            legs[name] = {"workload": ln["config"]["workload"], "metric": ln["metric"], "value": ln["value"], "unit": ln["unit"],
                          "ms_per_step": ln["ms_per_step"], "steps": ln["steps"], "parity": ln.get("parity"),
                          "roofline": {k2: rf.get(k2) for k2 in ("kernel", "achieved", "peak", "frac", "traffic", "algorithmic_bytes_per_launch")},
                          "gpu_launches": ln.get("gpu_launches"), "leg_wall_s": round(time.perf_counter() - t0, 1)}
            if name == "c5b":
                legs[name]["checkpoint_task_device_us"] = {m: v["device_us"] for m, v in ln["checkpoint_task"].items()}
                legs[name]["nop_round_trip_us"] = ln["trigger_latency"]["nop_round_trip_us"]
        except Exception as e:                                       # a failed leg must not take the headline line with it
            legs[name] = {"error": "%s: %s" % (type(e).__name__, e), "leg_wall_s": round(time.perf_counter() - t0, 1)}
        env.torch.cuda.empty_cache()
    return legs


def ring_on_region(cc, env, cur, shadow, P, k_exp, log_bytes, mutate, blocks_list=(1, 8, 32, 148), tasks=6):
    """CC_TASK_DELTA_CKPT on the workload's region through the ring buffer / persistent worker, at several worker
    footprints: device time per task from the %globaltimer stamps of the completion records.  (With a resident kernel
    only streams are synchronised, never the device: PAPER.md:L251.)"""
    torch, dev = env.torch, env.dev
    out = []
    log = torch.empty(log_bytes, dtype=torch.uint8, device=dev)
    for B in blocks_list:
        c2 = cc.Context(env.local, ring_capacity=16, worker_blocks=B, max_lifetime_ns=int(120e9))
        started = False
        try:
            c2.register_region(1, cur, P, shadow=shadow, snapshot_now=False)
            c2.log_attach(log)
            n = tasks if B > 1 else 2
            devms = []
            for t in range(n + 1):
                mutate(t)
                env.stream.synchronize()
                if t == 0:
                    c2.worker_start()
                    started = True
                r = c2.wait(c2.submit(cc.CC_TASK_DELTA_CKPT, region_id=1, epoch=t), 120.0)
                assert r.status == 0 and r.n_dirty == k_exp, r.as_dict()
                c2.wait(c2.submit(cc.CC_TASK_LOG_RESET), 10.0)
                if t:
                    devms.append((r.t_end_ns - r.t_start_ns) / 1e6)
            fp = c2.worker_footprint()
            out.append({"worker_blocks": fp["blocks"], "sm_share_pct": fp["sm_share_pct"], "threads_per_block": fp["threads_per_block"],
                        "registers_per_thread": fp["registers_per_thread"],
                        "device_ms_per_task": round(statistics.median(devms), 4), "tasks": len(devms)})
        finally:
            if started:
                c2.worker_stop()
            c2.shutdown()
    return {"what": "CC_TASK_DELTA_CKPT on this workload's region submitted through the ring (no kernel launch per boundary); "
                    "device time from the completion record's %globaltimer stamps; device log", "footprints": out}


# ------------------------------------------------------- generic timed checkpoints --

def timed_checkpoints(ctx, cc, env, rid, K, Wm, rearm, k_expect, cold, call=None, reset=True, phases=True, ahead=False):
    """W warm-ups, then K checkpoints of region `rid`, each timed on its own with CUDA events on the launch stream
    (re-arming the mutation and the optional L2 flush are NOT inside the events).  Returns per-step lists of ms:
    total, discovery (scan + compaction), writer (gather + commit + shadow), and the device time between the
    %globaltimer stamps of the result.
    phases=False: no event is recorded between the kernels of a call (an event there also keeps the kernels of the
    phases path from overlapping by programmatic dependent launch); discovery / writer are then 0.
    ahead=True: a ~150 us spin kernel is queued in front of the first event, so that the host has issued the whole call
    before the GPU reaches it -- the events then bracket GPU time only (an idle GPU would otherwise sit between the two
    events waiting for the interpreter to marshal the call, which is 10-20 us of a 60 us checkpoint)."""
    torch, stream = env.torch, env.stream
    res = cc.Result()
    call = call or (lambda it, res: ctx.checkpoint_delta(rid, it, res))
    tot, disc, wr, devt = [], [], [], []
    for it in range(Wm + K):
        rearm(it)
        if cold:
            env.flush_l2(it)
        evs = [env.ev() for _ in range(4)]
        torch.cuda.synchronize()
        if ahead:
            torch.cuda._sleep(300000)
        evs[0].record(stream)
        if phases:
            ctx.trace_events(evs[1], evs[2])
        call(it, res)
        evs[3].record(stream)
        torch.cuda.synchronize()
        if phases:
            ctx.trace_events(None, None)
        r = res.read()
        assert r.status == 0 and r.n_dirty == k_expect, (r.as_dict(), k_expect)
        if reset:
            ctx.log_reset()
        if it >= Wm:
            tot.append(evs[0].elapsed_time(evs[3]))
            disc.append(evs[0].elapsed_time(evs[2]) if phases else 0.0)
            wr.append(evs[2].elapsed_time(evs[3]) if phases else 0.0)
            devt.append((r.t_end_ns - r.t_start_ns) / 1e6)
    return tot, disc, wr, devt


def small_region_workload(args, env, name):
    """c1 / c3: 64 MiB regions.  They fit B200's L2 partly, so every timed checkpoint starts cold (512 MiB written in
    between, outside the events) and the warm number is reported beside it; HBM-fraction claims are made on c2 / c4."""
    import numpy as np
    import oracle
    import synth
    import paper_2606_23521_b200 as cc
    torch, dev, stream = env.torch, env.dev, env.stream
    K, Wm = args.steps, max(args.warmup, 3)
    if name == "c1":
        P, desc = 4096, "BASELINE.json configs[0]: 64 MiB raw bytes, 16,384 pages x 4 KiB, 1 % of the pages dirtied by 1-8 byte flips"
        cur = synth.raw_region(64 << 20, 1001 + env.rank, dev)
        old = cur.clone()
        pages = synth.mutate_byte_flips(cur, P, 0.01, 1001)           # the config's own mutation, for the parity leg
    else:
        P, desc = 65536, "BASELINE.json configs[2]: LoRA rank-16 A/B for q,k,v,o x 32 layers, fp32, 1,024 pages x 64 KiB, 5 % of the pages updated"
        cur = synth.lora_region(32, 1003 + env.rank, dev)
        old = cur.clone()
        pages = synth.lora_update(cur, P, 0.05, 1003)
    N = cur.numel()
    k = len(pages)
    n_pages = N // P
    ctx = cc.Context(env.local)
    shadow = ctx.register_region(1, cur, P, shadow=old.clone(), snapshot_now=False)
    cap = n_pages * (16 + P) + 32
    log = torch.zeros(cap, dtype=torch.uint8, device=dev)
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(log, committed)
    ctx.apply_attach(k + 64)
    res = cc.Result()
    # ---- parity (untimed): checkpoint + apply round trip against the oracle ----
    parity = None
    if not args.no_parity:
        ctx.checkpoint_delta(1, 7, res)
        torch.cuda.synchronize()
        r = res.read()
        olog = np.zeros(cap, np.uint8)
        osh = old.cpu().numpy().copy()
        st, D, nb, W = oracle.checkpoint(cur.cpu().numpy(), osh, P, 1, 7, olog, 0)
        assert (r.status, r.n_dirty, r.bytes) == (st, D.size, nb) and D.tolist() == pages.tolist() == ctx.dirty_list(1).tolist()
        assert np.array_equal(log.cpu().numpy()[:nb], olog[:nb]) and np.array_equal(shadow.cpu().numpy(), osh)
        new = cur.clone()
        cur.copy_(old)
        shadow.copy_(old)
        res.clear()
        ctx.apply_log(log, nb, res)
        torch.cuda.synchronize()
        r = res.read()
        host = old.cpu().numpy().copy()
        assert (r.status, r.n_dirty, r.bytes) == oracle.apply_log(olog, nb, [oracle.Region(1, P, host)])
        assert torch.equal(cur, new) and torch.equal(shadow, new) and np.array_equal(host, new.cpu().numpy())
        parity = {"checked": "dirty list, %d log bytes, shadow, and apply(old snapshot, log) == new region: bit-exact with the oracle" % nb,
                  "ok": True}
        ctx.log_reset()
    else:
        shadow.copy_(cur)
    # ---- timed: the same dirty set re-armed by toggling one byte per chosen page ----
    pg = pages.to(dev)
    offs = pg * P + (pg * 2654435761 % P)
    masks = torch.full((k,), 0x11, dtype=torch.uint8, device=dev)
    rearm = lambda it: synth.toggle_flips(cur, offs, masks)
    sampler = ClockSampler(env.local).start()
    launches0 = ctx.kernel_launches()
    env.barrier()
    tot, _, _, devt = timed_checkpoints(ctx, cc, env, 1, K, Wm, rearm, k, cold=True, phases=False, ahead=True)
    env.barrier()
    launches = (ctx.kernel_launches() - launches0) * K // (K + Wm)
    clocks = sampler.stop()
    tot_w, _, _, devt_w = timed_checkpoints(ctx, cc, env, 1, K, Wm, rearm, k, cold=False, phases=False, ahead=True)
    # the split into discovery / writer needs events between the kernels (which cost the kernels their overlap), and the
    # call issued to an idle GPU shows what the interpreter adds: both reported beside the headline, not in it
    tot_p, disc, wr, _ = timed_checkpoints(ctx, cc, env, 1, K, Wm, rearm, k, cold=True, phases=True, ahead=False)
    # ---- e2e: pinned host log, the mutation bytes come from host memory, result read on the host ----
    e2e = None
    if not args.no_e2e:
        hlog = torch.zeros(cap, dtype=torch.uint8, pin_memory=True)
        ctx.log_attach(hlog, committed)
        masks_host = masks.cpu().pin_memory()
        mstage = torch.empty_like(masks)
        times = []
        for it in range(Wm + K):
            env.flush_l2(it)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            mstage.copy_(masks_host, non_blocking=True)            # H2D: this step's new bytes
            synth.toggle_flips(cur, offs, mstage)
            ctx.checkpoint_delta(1, 100 + it, res)
            torch.cuda.synchronize()
            r = res.read()                                         # the result, read on the host
            if it >= Wm:
                times.append((time.perf_counter() - t0) * 1e3)
            assert r.status == 0 and r.n_dirty == k
            ctx.log_reset()
        e2e = {"ms": statistics.mean(times), "h2d": k, "d2h": k * (16 + P) + 32 + 64}
    ms = env.rmax(statistics.mean(tot))
    if env.rank == 0:
        algo = 2 * N + 3 * k * P
        line = base_line(env, K, Wm, env.world * N / (ms * 1e-3) / 1e9, ms, desc + "; log in device memory",
                         {"page_bytes": P, "region_bytes_per_gpu": N, "dirty_pages": k, "dirty_bytes": k * P,
                          "l2": "flushed: 512 MiB written between timed iterations (outside the events); each step timed on its own",
                          "timing": "CUDA events around each cc_checkpoint_delta, the call queued behind a 150 us spin kernel so that the "
                                    "events bracket GPU time only; the re-arming byte flips and the flush are not timed"},
                         "u8 (bitwise compare/copy; CRC32C in u32)")
        line["gpu_launches"] = int(launches)
        line["clocks"] = clocks
        line["parity"] = parity
        line["phases_ms"] = {"checkpoint_total": round(ms, 4), "best_checkpoint_total": round(min(tot), 4),
                             "device_stamps_total": round(statistics.mean(devt), 4),
                             "warm_l2_checkpoint_total": round(statistics.mean(tot_w), 4), "warm_l2_best": round(min(tot_w), 4),
                             "warm_l2_device_stamps_total": round(statistics.mean(devt_w), 4),
                             "issued_to_idle_gpu_with_events_between_kernels": {
                                 "total": round(statistics.mean(tot_p), 4), "discovery": round(statistics.mean(disc), 4),
                                 "writer": round(statistics.mean(wr), 4)}}
        line["roofline"] = roofline("cc_checkpoint_delta (whole call: launch- and latency-bound at this size)", algo, ms, name,
                                    kernels=("cc_scan_kernel", "cc_small_tail_kernel"))
        line["roofline"]["note"] = "64 MiB regions are launch/latency-bound, not HBM-bound; HBM-fraction claims are made on c2 / c4"
        if e2e:
            line["e2e"] = {"value": round(env.world * N / (e2e["ms"] * 1e-3) / 1e9, 2), "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"],
                           "d2h_bytes_per_step": e2e["d2h"], "ms_per_step": round(e2e["ms"], 4),
                           "path": "cc_checkpoint_delta storing straight into a pinned host log; host wall clock per step incl. H2D of the "
                                   "new bytes, launch, synchronize and reading the result"}
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = oracle_leg(name, args)
        emit(args, line)
    ctx.shutdown()


# ------------------------------------------------------------------------ c4 --

def _fit_gib(torch, want, copies, extra_gib=6):
    free, _ = torch.cuda.mem_get_info()
    g = want
    while g > 1 and copies * (g << 30) + (extra_gib << 30) > free:
        g //= 2
    return g


def run_c4_sparse(args, env):
    import numpy as np
    import oracle
    import synth
    import paper_2606_23521_b200 as cc
    torch, dev = env.torch, env.dev
    K, Wm = args.steps, max(args.warmup, 3)
    gib = _fit_gib(torch, args.large_gib, 2)
    N = gib << 30
    cur = synth.bf16_normal_region(N, 1004 + env.rank, dev)
    shadow = torch.empty_like(cur)
    for o in range(0, N, 1 << 30):
        shadow[o:o + (1 << 30)] = cur[o:o + (1 << 30)]
    Ps = (65536, 16384, 4096)
    ctx = cc.Context(env.local)
    for i, P in enumerate(Ps):
        ctx.register_region(i + 1, cur, P, shadow=shadow, snapshot_now=False)     # one memory, three page sizes
    sweep = {}
    parity = None
    clocks = None
    launches = 0
    for i, P in enumerate(Ps):
        rid = i + 1
        pages, offs, masks = synth.sparse_xor_flips(cur, P, 0.001, 1004 + P)
        k = len(pages)
        log = torch.zeros(k * (16 + P) + 32, dtype=torch.uint8, device=dev)
        ctx.log_attach(log)
        if not args.no_parity and env.rank == 0:
            # untimed: the whole checkpoint against the oracle, chunk by chunk (host RAM cannot hold 2 x 64 GiB)
            from oracle import chunked
            o_cpu, m_cpu = offs.cpu().numpy(), masks.cpu().numpy()

            def fetch_shadow0(o, n):
                a = cur[o:o + n].cpu().numpy()
                lo, hi = np.searchsorted(o_cpu, [o, o + n])
                a[o_cpu[lo:hi] - o] ^= m_cpu[lo:hi]
                return a
            res = cc.Result()
            ctx.checkpoint_delta(rid, 5, res)
            torch.cuda.synchronize()
            r = res.read()
            kk, nb, D = chunked.verify_checkpoint_chunked(N, P, rid, 5, lambda o, n: cur[o:o + n].cpu().numpy(), fetch_shadow0,
                                                          lambda o, n: log[o:o + n].cpu().numpy(), chunk_bytes=1 << 30, threads=16)
            assert (r.status, r.n_dirty, r.bytes) == (0, kk, nb) and D.tolist() == pages.tolist() == ctx.dirty_list(rid).tolist()
            assert all(torch.equal(shadow[o:o + (1 << 30)], cur[o:o + (1 << 30)]) for o in range(0, N, 1 << 30))
            parity = parity or {"checked": [], "ok": True}
            parity["checked"].append("%d KiB pages: dirty list (%d pages), all %d log bytes, shadow == region: bit-exact with "
                                     "oracle.checkpoint run on every 1 GiB chunk of the %d GiB region" % (P >> 10, kk, nb, gib))
            ctx.log_reset()
        else:
            synth.toggle_flips(shadow, offs, masks)                # shadow := cur
        if P == Ps[0]:
            sampler = ClockSampler(env.local).start()
            launches0 = ctx.kernel_launches()
        env.barrier()
        tot, disc, wr, _ = timed_checkpoints(ctx, cc, env, rid, K if P == Ps[0] else max(3, K // 4), Wm,
                                          lambda it: synth.toggle_flips(cur, offs, masks), k, cold=False)
        env.barrier()
        if P == Ps[0]:
            clocks = sampler.stop()
            launches = (ctx.kernel_launches() - launches0) * K // (K + Wm)
        ms, dms = statistics.mean(tot), statistics.mean(disc)
        sweep["%dKiB" % (P >> 10)] = {"dirty_pages": k, "ms_total": round(ms, 4), "ms_scan_compact": round(dms, 4),
                                      "ms_writer": round(statistics.mean(wr), 4), "best_ms_total": round(min(tot), 4),
                                      "region_GBps": round(N / ms / 1e6, 1),
                                      "hbm_GBps_2N_3kP": round((2 * N + 3 * k * P) / ms / 1e6, 1),
                                      "scan_GBps_2N": round(2 * N / dms / 1e6, 1)}
        del log
    P = Ps[0]
    head = sweep["64KiB"]
    ms = env.rmax(head["ms_total"])
    if env.rank == 0:
        line = base_line(env, K, Wm, env.world * N / (ms * 1e-3) / 1e9, ms,
                         "BASELINE.json configs[3], sparse sweep: %d GiB bf16 region, 0.1 %% of the pages dirty, 64 KiB pages "
                         "(value); page sizes 4 / 16 / 64 KiB in page_size_sweep; log in device memory" % gib,
                         {"page_bytes": P, "region_bytes_per_gpu": N, "dirty_pages": head["dirty_pages"],
                          "l2": "inputs larger than L2 (2 x %d GiB streamed per step)" % gib,
                          "capacity": "full size" if gib == args.large_gib else "region halved to %d GiB to fit region + shadow (SURVEY.md 8d fallback ii)" % gib,
                          "timing": "CUDA events around each cc_checkpoint_delta; the re-arming byte flips are not timed"},
                         "u8 (bitwise compare/copy of bf16 bytes; CRC32C in u32)")
        line["gpu_launches"] = int(launches)
        line["clocks"] = clocks
        line["parity"] = parity
        line["page_size_sweep"] = sweep
        line["roofline"] = roofline("cc_scan_kernel", 2 * N, head["ms_scan_compact"], args.workload)
        line["roofline"]["note"] = "duration = scan + compaction (events after the compaction kernel); the compaction is ~0.02 ms of it"
        if not args.no_e2e:
            line["e2e"] = c4_e2e(args, env, ctx, cc, cur, shadow, Ps[0], 1, sparse=True)
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = oracle_leg("c4-sparse", args)
        print(json.dumps(line), flush=True)
    ctx.shutdown()


def c4_e2e(args, env, ctx, cc, cur, shadow, P, rid, sparse):
    """Sparse: pinned host log, the flip bytes copied H2D, result read on the host."""
    import synth
    torch, dev = env.torch, env.dev
    N = cur.numel()
    pages, offs, masks = synth.sparse_xor_flips(cur, P, 0.001, 99 + P)
    k = len(pages)
    synth.toggle_flips(shadow, offs, masks)
    hlog = torch.zeros(k * (16 + P) + 32, dtype=torch.uint8, pin_memory=True)
    ctx.log_attach(hlog)
    mh = masks.cpu().pin_memory()
    mst = torch.empty_like(masks)
    res = cc.Result()
    K = max(3, args.steps // 4)
    times = []
    for it in range(2 + K):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        mst.copy_(mh, non_blocking=True)
        synth.toggle_flips(cur, offs, mst)
        ctx.checkpoint_delta(rid, 300 + it, res)
        torch.cuda.synchronize()
        r = res.read()
        if it >= 2:
            times.append((time.perf_counter() - t0) * 1e3)
        assert r.status == 0 and r.n_dirty == k
        ctx.log_reset()
    ms = statistics.mean(times)
    return {"value": round(env.world * N / (ms * 1e-3) / 1e9, 2), "unit": UNIT, "h2d_bytes_per_step": k,
            "d2h_bytes_per_step": k * (16 + P) + 32 + 64, "ms_per_step": round(ms, 4),
            "path": "cc_checkpoint_delta storing straight into a pinned host log (64 KiB pages); host wall clock per step incl. "
                    "H2D of the new bytes, launch, synchronize and reading the result"}


def _tests_util():
    """The C4 all-dirty checker lives with the tests (tests/gpu_util.py: it calls oracle/chunked.py); the untimed parity
    legs below borrow it from there."""
    tdir = os.path.join(ROOT, "tests")
    if tdir not in sys.path:
        sys.path.insert(0, tdir)
    import gpu_util
    return gpu_util


def run_c4_full(args, env):
    import synth
    import paper_2606_23521_b200 as cc
    torch, dev = env.torch, env.dev
    K, Wm = max(3, args.steps // 4), 3
    gib = _fit_gib(torch, args.large_gib, 3.02)
    N = gib << 30
    cur = synth.bf16_normal_region(N, 1004 + env.rank, dev)
    Ps = (65536, 16384, 4096)
    sweep, parity, clocks, launches = {}, None, None, 0
    for P in Ps:
        n_pages = N // P
        ctx = cc.Context(env.local)
        shadow = ctx.register_region(1, cur, P)
        log = torch.empty(n_pages * (16 + P) + 32, dtype=torch.uint8, device=dev)
        ctx.log_attach(log)
        offs, masks = synth.all_dirty_flips(N, P, 1004 + P, dev)
        if not args.no_parity and env.rank == 0:
            synth.toggle_flips(cur, offs, masks)
            res = cc.Result()
            ctx.checkpoint_delta(1, 6, res)
            torch.cuda.synchronize()
            r = res.read()
            kk, nb, D = _tests_util().verify_all_dirty(cur, log, offs, masks, P, 1, 6)
            assert (r.status, r.n_dirty, r.bytes) == (0, n_pages, nb) and kk == n_pages
            assert all(torch.equal(shadow[o:o + (1 << 30)], cur[o:o + (1 << 30)]) for o in range(0, N, 1 << 30))
            parity = parity or {"checked": [], "ok": True}
            parity["checked"].append("%d KiB pages: all %d records (header, CRC32C, payload) and the commit record of the %d GiB "
                                     "device log: bit-exact with oracle.checkpoint run on every 1 GiB chunk; shadow == region"
                                     % (P >> 10, kk, gib))
            ctx.log_reset()
        if P == Ps[0]:
            sampler = ClockSampler(env.local).start()
            launches0 = ctx.kernel_launches()
        env.barrier()
        tot, disc, wr, _ = timed_checkpoints(ctx, cc, env, 1, K, Wm, lambda it: synth.toggle_flips(cur, offs, masks), n_pages, cold=False)
        env.barrier()
        if P == Ps[0]:
            clocks = sampler.stop()
            launches = (ctx.kernel_launches() - launches0) * K // (K + Wm)
        totf, _, _, _ = timed_checkpoints(ctx, cc, env, 1, K, 2, lambda it: synth.toggle_flips(cur, offs, masks), n_pages, cold=False,
                                       call=lambda it, res: ctx.checkpoint_delta_fused(1, it, res))
        ms = statistics.mean(tot)
        sweep["%dKiB" % (P >> 10)] = {"dirty_pages": n_pages, "ms_total": round(ms, 4), "ms_scan_compact": round(statistics.mean(disc), 4),
                                      "ms_writer": round(statistics.mean(wr), 4), "best_ms_total": round(min(tot), 4),
                                      "region_GBps": round(N / ms / 1e6, 1), "dirty_GBps_writer": round(N / statistics.mean(wr) / 1e6, 1),
                                      "writer_hbm_GBps_3kP": round(3 * N / statistics.mean(wr) / 1e6, 1),
                                      "hbm_GBps_2N_3kP": round(5 * N / ms / 1e6, 1),
                                      "fused_single_pass_ms_total": round(statistics.mean(totf), 4)}
        ctx.shutdown()
        del log, shadow
        torch.cuda.empty_cache()
    head = sweep["64KiB"]
    ms = env.rmax(head["ms_total"])
    e2e = None
    if not args.no_e2e and env.rank == 0:
        import gc
        del cur, offs, masks
        gc.collect()
        torch.cuda.empty_cache()
        e2e = c4_full_arena(args, env, cc, 65536, verify=not args.no_parity)
        if parity and e2e.get("parity"):
            parity["checked"].append(e2e.pop("parity"))
    if env.rank == 0:
        line = base_line(env, K, Wm, env.world * N / (ms * 1e-3) / 1e9, ms,
                         "BASELINE.json configs[3], 100 %% dirty sweep: every page of a %d GiB bf16 region dirty (one flipped byte per page), "
                         "64 KiB pages (value); 4 / 16 / 64 KiB in page_size_sweep; log in device memory" % gib,
                         {"page_bytes": 65536, "region_bytes_per_gpu": N, "dirty_pages": head["dirty_pages"],
                          "l2": "inputs larger than L2",
                          "capacity": "SURVEY.md 8d fallback (ii): %d GiB is the largest power-of-two slice whose %d GiB device log fits beside "
                                      "region and shadow in 180 GB; the full 64 GiB arena runs as e2e through one pinned host log (fallback i)" % (gib, gib),
                          "timing": "CUDA events around each cc_checkpoint_delta; the re-arming byte flips are not timed"},
                         "u8 (bitwise compare/copy of bf16 bytes; CRC32C in u32)")
        line["gpu_launches"] = int(launches)
        line["clocks"] = clocks
        line["parity"] = parity
        line["page_size_sweep"] = sweep
        line["roofline"] = roofline("cc_gather_kernel", 3 * N, head["ms_writer"], args.workload)
        if e2e:
            line["e2e"] = e2e
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = oracle_leg("c4-full", args)
        print(json.dumps(line), flush=True)


def c4_full_arena(args, env, cc, P, verify, regions=8, region_gib=8):
    """SURVEY.md 8d capacity fallback (i): the 64 GiB arena as 8 x 8 GiB regions, every page dirty, checkpointed one after
    the other into ONE pinned host log of 8.1 GiB that the harness verifies (untimed) and resets between regions --
    the link-bound worst case config 4 is about."""
    import synth
    torch, dev = env.torch, env.dev
    R = region_gib << 30
    free, _ = torch.cuda.mem_get_info()
    while regions > 1 and 2 * regions * R + (4 << 30) > free:
        regions //= 2
    arena = synth.bf16_normal_region(regions * R, 1004, dev)
    ctx = cc.Context(env.local)
    shadows = []
    for i in range(regions):
        shadows.append(ctx.register_region(i + 1, arena[i * R:(i + 1) * R], P))
    n_pages = R // P
    cap = n_pages * (16 + P) + 32
    hlog = torch.empty(cap, dtype=torch.uint8, pin_memory=True)
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(hlog, committed)
    res = cc.Result()
    flips = [synth.all_dirty_flips(R, P, 7000 + i, dev) for i in range(regions)]
    times, ok = [], 0
    for rnd in range(2):                                             # round 0 warms up and verifies; round 1 is timed
        for i in range(regions):
            v = arena[i * R:(i + 1) * R]
            synth.toggle_flips(v, *flips[i])
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ctx.checkpoint_delta(i + 1, 10 * rnd + i, res)
            torch.cuda.synchronize()
            r = res.read()
            dt = (time.perf_counter() - t0) * 1e3
            assert r.status == 0 and r.n_dirty == n_pages and r.bytes == cap and int(committed.item()) == cap, r.as_dict()
            if rnd == 0 and verify:
                kk, nb, D = _tests_util().verify_all_dirty(v, hlog, flips[i][0], flips[i][1], P, i + 1, i, log_is_host=True)
                assert kk == n_pages and nb == cap and torch.equal(shadows[i], v)
                ok += 1
            if rnd == 1:
                times.append(dt)
            ctx.log_reset()                                         # the harness has consumed the log: rewind
    ctx.shutdown()
    total = sum(times)
    out = {"value": round(regions * R / (total * 1e-3) / 1e9, 2), "unit": UNIT, "h2d_bytes_per_step": 0,
           "d2h_bytes_per_step": regions * cap + 64 * regions, "ms_per_step": round(total, 3),
           "host_link_GBps_log": round(regions * cap / (total * 1e-3) / 1e9, 2),
           "path": "SURVEY.md 8d fallback (i): the %d GiB arena as %d x %d GiB regions (%d KiB pages, every page dirty), "
                   "cc_checkpoint_delta of each into ONE pinned %.1f GiB host log, result read on the host and the log rewound "
                   "between regions; one step = the whole arena; host wall clock; link-bound (SM stores cap at 52.7 GB/s)"
                   % (regions * region_gib, regions, region_gib, P >> 10, cap / 2**30)}
    if verify:
        out["parity"] = ("arena: all %d x %d records of the pinned host log and the shadows bit-exact with the oracle (chunk-wise), %d regions"
                         % (ok, n_pages, ok))
    return out


# ------------------------------------------------------------------------ c5a --

def run_c5a(args, env):
    import numpy as np
    import oracle
    import synth
    import paper_2606_23521_b200 as cc
    torch, dev, stream = env.torch, env.dev, env.stream
    K, Wm = args.steps, max(args.warmup, 3)
    arena_bytes = 8 << 30
    olog, W, n_rec, views = build_c5a_log(arena_bytes)
    arena0 = synth.raw_region(arena_bytes, 1005, dev)
    work = arena0.clone()
    ctx = cc.Context(env.local)
    for rid, (o, sz, P) in views.items():
        ctx.register_region(rid, work[o:o + sz], P)
    ctx.apply_attach(n_rec + 128)
    log_dev = torch.from_numpy(olog[:W]).to(dev)
    log_pin = torch.from_numpy(olog[:W]).pin_memory()
    res = cc.Result()
    parity = None
    if not args.no_parity:
        host = arena0.cpu().numpy()
        exp = oracle.apply_log(olog, W, [oracle.Region(rid, P, host[o:o + sz]) for rid, (o, sz, P) in views.items()])
        for name, lg in (("device log", log_dev), ("pinned host log", log_pin)):
            work.copy_(arena0)
            res.clear()
            ctx.apply_log(lg, W, res)
            torch.cuda.synchronize()
            r = res.read()
            assert (r.status, r.n_dirty, r.bytes) == exp and r.epoch == 100, (r.as_dict(), exp)
            assert all(np.array_equal(work[o:o + (1 << 30)].cpu().numpy(), host[o:o + (1 << 30)]) for o in range(0, arena_bytes, 1 << 30)), name
        parity = {"checked": "the 8 GiB arena after cc_apply_log (from a device log and from a pinned host log) == the arena after "
                             "oracle.apply_log, byte for byte; %d records, %d log bytes written by the oracle's record writer" % (n_rec, W),
                  "ok": True}
        del host

    def timed(lg, n, warm):
        ts = []
        for it in range(warm + n):
            work[:1 << 20].zero_()                                   # something to repair; the log's pages are rewritten anyway
            torch.cuda.synchronize()
            e0 = env.ev()
            ctx.apply_log(lg, W, res)
            e1 = env.ev()
            torch.cuda.synchronize()
            r = res.read()
            assert r.status == 0 and r.bytes == W
            if it >= warm:
                ts.append(e0.elapsed_time(e1))
        return ts
    sampler = ClockSampler(env.local).start()
    launches0 = ctx.kernel_launches()
    env.barrier()
    t_dev = timed(log_dev, K, Wm)
    env.barrier()
    launches = (ctx.kernel_launches() - launches0) * K // (K + Wm)
    clocks = sampler.stop()
    ms = env.rmax(statistics.mean(t_dev))
    e2e = None
    if not args.no_e2e:
        ctx.apply_stage_attach(W)
        t_pin = timed(log_pin, max(3, K // 2), 2)
        ctx.apply_stage_attach(0)
        t_pin2 = timed(log_pin, 3, 1)
        e2e = (statistics.mean(t_pin), statistics.mean(t_pin2))
    if env.rank == 0:
        algo = 3 * W                                                 # the method's own bytes: the log read once, live page + shadow written
        line = base_line(env, K, Wm, env.world * W / (ms * 1e-3) / 1e9, ms,
                         "BASELINE.json configs[4], recovery half: replay of a committed log of %d page records in 100 epochs (mixed 4 / 16 / 64 KiB "
                         "pages, %d bytes, written by the oracle's record writer) into an 8 GiB arena registered as three regions; log in "
                         "device memory; value = log GB/s replayed" % (n_rec, W),
                         {"log_bytes": W, "page_records": n_rec, "epochs": 100, "arena_bytes": arena_bytes,
                          "l2": "the log (284 MB) and the touched pages exceed L2 (126 MB)",
                          "timing": "CUDA events around each cc_apply_log"},
                         "u8 (byte copy; CRC32C in u32)")
        line["metric"] = METRICS["c5a"]
        line["gpu_launches"] = int(launches)
        line["clocks"] = clocks
        line["parity"] = parity
        line["phases_ms"] = {"apply_total": round(ms, 4), "best": round(min(t_dev), 4), "records_per_s": round(n_rec / (ms * 1e-3))}
        line["roofline"] = roofline("cc_apply_* (whole replay: parse + validate + scatter)", algo, ms, "c5a", kernels=("cc_apply_*",))
        line["roofline"]["note"] = ("algorithmic bytes = 3 x log bytes (SURVEY.md 8d: the method reads the log once and writes every payload byte to the "
                                    "live page and to the shadow); the implementation reads the log three times (candidate search, validation, "
                                    "scatter) -- that shows in `traffic`, not here")
        if e2e:
            line["e2e"] = {"value": round(env.world * W / (e2e[0] * 1e-3) / 1e9, 2), "unit": UNIT, "h2d_bytes_per_step": W,
                           "d2h_bytes_per_step": 64, "ms_per_step": round(e2e[0], 4),
                           "path": "cc_apply_log from a PINNED HOST log with a device staging buffer attached (one copy-engine pass over "
                                   "the host link, H2D DMA peak 55.6 GB/s => floor %.2f ms); result read on the host" % (W / 55.6e6),
                           "ms_without_stage_buffer": round(e2e[1], 4)}
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = oracle_leg("c5a", args)
        emit(args, line)
    ctx.shutdown()


# ------------------------------------------------------------------------ c5b --

def _pct(xs, q):
    xs = sorted(xs)
    return xs[min(len(xs) - 1, int(q * len(xs)))]


def run_c5b(args, env):
    import ctypes
    import numpy as np
    import oracle
    import synth
    import paper_2606_23521_b200 as cc
    torch, dev = env.torch, env.dev
    P, n_pages, n_mut, n_tasks = 4096, 65536, 656, args.tasks
    N = P * n_pages
    cur = synth.raw_region(N, 1006, dev)
    per = n_mut * (16 + P) + 32
    worst = n_pages * (16 + P) + 32
    A = 2 * ((1006 * 7919 + 12345) % 100000) + 1
    host_cur = cur.cpu().numpy().copy()
    host_sh = host_cur.copy()
    n_parity = 0 if args.no_parity else 32
    out = {}
    launches_total = 0
    for mode, flags in (("three_phase", 0), ("fused", cc.CC_TASKF_FUSED)):
        # latency configuration: every co-resident worker CTA (the default footprint, CC_WORKER_BLOCKS_DEFAULT = 16 CTAs,
        # trades task time for SMs left to the application: see --workload overlap)
        ctx = cc.Context(env.local, ring_capacity=256, worker_blocks=cc.CC_WORKER_BLOCKS_ALL, max_lifetime_ns=int(300e9))
        sh = ctx.register_region(1, cur, P)
        log = torch.zeros(1 << 30, dtype=torch.uint8, pin_memory=True)
        ctx.log_attach(log)
        lib, h = ctx.lib, ctx.h
        seq = ctypes.c_uint64()
        r = cc.cc_result()
        # host-launched comparison + launch cost (before the worker occupies the SMs)
        res = cc.Result()
        idx = (torch.arange(n_mut, device=dev) * A % n_pages) * P
        host_launched = []
        for i in range(30):
            cur[idx] ^= 0x5A
            torch.cuda.synchronize()
            t0 = time.perf_counter_ns()
            (ctx.checkpoint_delta_fused if flags else ctx.checkpoint_delta)(1, i, res)
            torch.cuda.synchronize()
            host_launched.append(time.perf_counter_ns() - t0)
            ctx.log_reset()
        if mode == "three_phase":
            launch_sync_ns, launch_batched_ns = ctx.measure_launch_cost(2000)
        host_cur = cur.cpu().numpy().copy()                          # shadow == region after the last checkpoint
        host_sh = host_cur.copy()
        olog = np.zeros(max(n_parity, 1) * per, dtype=np.uint8)
        Wo = 0
        ctx.worker_start()
        try:
            if mode == "three_phase":
                task = cc.cc_task(cc.CC_TASK_NOP, 0, 0, 0, 0, 0, 0, 0, 0, 0)
                submit_ns, nop_rt = [], []
                for i in range(2000):
                    t0 = time.perf_counter_ns()
                    lib.cc_submit(h, ctypes.byref(task), ctypes.byref(seq))
                    t1 = time.perf_counter_ns()
                    lib.cc_wait(h, seq.value, int(5e9), ctypes.byref(r))
                    t2 = time.perf_counter_ns()
                    submit_ns.append(t1 - t0)
                    nop_rt.append(t2 - t0)
                native_submit_ns = ctx.measure_submit_cost(200000)
                footprint = ctx.worker_footprint()
            rt, dev_ns = [], []
            ctx.wait(ctx.submit(cc.CC_TASK_LOG_RESET), 30.0)
            used = 0
            t_begin = time.perf_counter()
            for t in range(n_tasks):
                if used + max(per, worst if flags else 0) > log.numel() or t == n_parity:
                    if t == n_parity and n_parity:
                        assert np.array_equal(log.numpy()[:Wo], olog[:Wo]), "ring-task log differs from the oracle"
                    ctx.wait(ctx.submit(cc.CC_TASK_LOG_RESET), 30.0)
                    used = 0
                used += per
                pages, hh = synth.worker_mutation_pages(t, n_pages, n_mut, 1006)
                ctx.wait(ctx.submit(cc.CC_TASK_TEST_MUTATE, region_id=1, arg0=n_mut, arg1=A, arg2=hh), 30.0)
                ck = cc.cc_task(cc.CC_TASK_DELTA_CKPT, 1, flags, 0, 0, t, 0, 0, 0, 0)
                t0 = time.perf_counter_ns()
                lib.cc_submit(h, ctypes.byref(ck), ctypes.byref(seq))
                lib.cc_wait(h, seq.value, int(30e9), ctypes.byref(r))
                t1 = time.perf_counter_ns()
                rt.append(t1 - t0)
                dev_ns.append(r.t_end_ns - r.t_start_ns)
                assert r.status == 0 and r.n_dirty == n_mut, (t, r.as_dict())
                if t < n_parity:
                    for j, p in enumerate(pages):
                        host_cur[p * P + (hh + j) % P] ^= 0x5A
                    st, D, nb, Wo = oracle.checkpoint(host_cur, host_sh, P, 1, t, olog, Wo)
                    assert st == 0 and D.size == n_mut and r.log_offset_after == Wo
            wall = time.perf_counter() - t_begin
        finally:
            ctx.worker_stop()
        launches_total += ctx.kernel_launches()
        torch.cuda.synchronize()
        assert torch.equal(sh, cur)
        us = lambda xs, q: round(_pct(xs, q) / 1e3, 2)
        out[mode] = {"round_trip_us": {"p50": us(rt, 0.5), "p99": us(rt, 0.99)}, "device_us": {"p50": us(dev_ns, 0.5), "p99": us(dev_ns, 0.99)},
                     "host_launched_same_checkpoint_us": {"p50": us(host_launched, 0.5), "p99": us(host_launched, 0.99)},
                     "wall_s_for_all_tasks_incl_mutation_tasks": round(wall, 3), "dev_ns_mean": statistics.mean(dev_ns)}
        ctx.shutdown()
        del log
    if env.rank == 0:
        best = "fused" if out["fused"]["dev_ns_mean"] <= out["three_phase"]["dev_ns_mean"] else "three_phase"
        ms = out[best]["dev_ns_mean"] / 1e6
        for m in out.values():
            m.pop("dev_ns_mean")
        us = lambda xs, q: round(_pct(xs, q) / 1e3, 2)
        line = base_line(env, n_tasks, 0, N / (ms * 1e-3) / 1e9, ms,
                         "BASELINE.json configs[4], worker half: %d checkpoint tasks submitted through the ring buffer to the persistent worker on a "
                         "256 MiB region (65,536 x 4 KiB pages), 656 pages (1 %%) dirtied before every task (CC_TASK_TEST_MUTATE); pinned host log; "
                         "value = region GB/s from the mean device time of the %s task" % (n_tasks, best),
                         {"page_bytes": P, "region_bytes_per_gpu": N, "dirty_pages": n_mut, "bytes_per_task": per,
                          "l2": "the region (2 x 256 MiB read per task) exceeds L2 (126 MB); tasks run back to back",
                          "timing": "device time = %globaltimer stamps in the completion record; round trip = host clock around cc_submit + cc_wait"},
                         "u8 (bitwise compare/copy; CRC32C in u32)")
        line["metric"] = METRICS["c5b"]
        line["gpu_launches"] = int(launches_total)
        line["gpu_launches_note"] = "host-launched comparison legs + ONE persistent worker launch per mode; the %d ring tasks launch nothing" % n_tasks
        line["parity"] = None if args.no_parity else {"checked": "log bytes of the first %d ring tasks of each mode == the oracle's (mutation replayed in closed form); "
                                                                 "k == 656 and status on all %d tasks of both modes; shadow == region at the end" % (n_parity, n_tasks), "ok": True}
        line["trigger_latency"] = {"submit_host_cost_us_through_ctypes": {"p50": us(submit_ns, 0.5), "p99": us(submit_ns, 0.99)},
                                   "submit_host_cost_native_ns": round(native_submit_ns, 1),
                                   "nop_round_trip_us": {"p50": us(nop_rt, 0.5), "p99": us(nop_rt, 0.99)},
                                   "empty_kernel_launch_us": {"sync_each": round(launch_sync_ns / 1e3, 2), "batched": round(launch_batched_ns / 1e3, 2)},
                                   "paper_context": "Table 7 (RTX PRO 6000): ring submit < 0.1 us, cudaLaunchKernel 7.6 us sync / 2.5 us batch; "
                                                    "round trip ~80 us for a trivial op (L307)"}
        line["checkpoint_task"] = out
        line["worker_footprint"] = footprint
        line["roofline"] = roofline("cc_worker_kernel (one %s checkpoint task)" % best, 2 * N + 3 * n_mut * P, ms, "c5b", kernels=("cc_pass_kernel",))
        line["roofline"]["traffic_note"] = ("traffic is that of the host-launched equivalent of the fused task (cc_pass_kernel on the same region and "
                                            "pinned log): a never-ending worker kernel cannot be profiled launch by launch")
        line["e2e"] = {"value": round(N / (out[best]["round_trip_us"]["p50"] * 1e-6) / 1e9, 2), "unit": UNIT,
                       "h2d_bytes_per_step": 64, "d2h_bytes_per_step": per + 64, "ms_per_step": round(out[best]["round_trip_us"]["p50"] / 1e3, 4),
                       "path": "host clock around cc_submit + cc_wait (p50): the 64-byte descriptor crosses the host link, the records go "
                               "straight into the pinned host log, the 64-byte completion record is read on the host"}
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = oracle_leg("c5b", args)
        emit(args, line)


# -------------------------------------------------------------------- overlap --

def run_overlap(args, env):
    """Checkpointing next to compute (Fig. 7b "Throughput impact with overlapped delta checkpointing"; L427 "The
    persistent kernel occupies 1 block out of 188 SMs = 0.53% of GPU resources").  For each worker footprint B
    (persistent CTAs out of 148 SMs): a bandwidth-bound application kernel (torch device-to-device copy of 4 GiB, read + write
    bytes) while the worker idles, the device time of one delta-checkpoint task (256 MiB region, 1 % dirty 4 KiB pages, device
    log), and both at the same time.  Second part: 48 small regions at one boundary, cc_checkpoint_all against a loop."""
    import paper_2606_23521_b200 as cc
    torch, dev, stream = env.torch, env.dev, env.stream
    P, N = 4096, 256 << 20
    n_pages = N // P
    n_mut = math.ceil(0.01 * n_pages)
    A = 2 * ((1006 * 7919 + 12345) % 100000) + 1
    g = torch.Generator(device=dev)
    g.manual_seed(1006)
    cur = torch.randint(0, 256, (N,), dtype=torch.uint8, device=dev, generator=g)
    src = torch.empty(4 << 30, dtype=torch.uint8, device=dev)
    dst = torch.empty_like(src)
    per = n_mut * (16 + P) + 32

    def copy_gbps(reps=6):
        stream.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            dst.copy_(src)
        e1.record(stream)
        e1.synchronize()
        return 2 * src.numel() * reps / (e0.elapsed_time(e1) * 1e-3) / 1e9

    base = copy_gbps()
    rows = []
    for B in (1, 2, 4, 8, 16, 32, 64):
        ctx = cc.Context(env.local, ring_capacity=256, worker_blocks=B, max_lifetime_ns=int(120e9))
        ctx.register_region(1, cur, P)
        log = torch.empty(64 * per, dtype=torch.uint8, device=dev)
        ctx.log_attach(log)
        stream.synchronize()
        ctx.worker_start()
        row = {"worker_blocks": B, "sm_share_pct": ctx.worker_footprint()["sm_share_pct"]}
        print("overlap: worker_blocks", B, file=sys.stderr, flush=True)
        try:
            row["copy_alone_GBps"] = round(copy_gbps(), 1)

            def tasks(n, flags):
                seqs = []
                for t in range(n):
                    hh = (1006 * 2654435761 + t * 40503) & 0xFFFFFFFF
                    ctx.submit(cc.CC_TASK_TEST_MUTATE, region_id=1, arg0=n_mut, arg1=A, arg2=hh)
                    seqs.append(ctx.submit(cc.CC_TASK_DELTA_CKPT, region_id=1, epoch=t, flags=flags))
                return seqs

            def collect(seqs):
                rs = [ctx.wait(s, 60.0) for s in seqs]
                assert all(r.status == 0 and r.n_dirty == n_mut for r in rs)
                ctx.wait(ctx.submit(cc.CC_TASK_LOG_RESET), 60.0)
                return statistics.median([(r.t_end_ns - r.t_start_ns) / 1e6 for r in rs])

            collect(tasks(4, 0))
            row["ckpt_alone_ms"] = round(collect(tasks(16, 0)), 4)
            n_tasks = min(60, max(8, int(6 * 2 * src.numel() / 6.0e12 * 1e3 / max(row["ckpt_alone_ms"], 1e-3)) + 4))
            seqs = tasks(n_tasks, 0)
            row["copy_with_ckpt_GBps"] = round(copy_gbps(), 1)
            row["ckpt_with_copy_ms"] = round(collect(seqs), 4)
            row["copy_loss_pct_idle_worker"] = round(100 * (1 - row["copy_alone_GBps"] / base), 1)
            row["copy_loss_pct_busy_worker"] = round(100 * (1 - row["copy_with_ckpt_GBps"] / base), 1)
        finally:
            ctx.worker_stop()
        ctx.shutdown()
        rows.append(row)
    # ---- many small regions at one boundary ----
    R, small_bytes, sp = 48, 4 << 20, 65536
    regs = [torch.randint(0, 256, (small_bytes,), dtype=torch.uint8, device=dev, generator=g) for _ in range(R)]
    ctx = cc.Context(env.local)
    for i, t in enumerate(regs):
        ctx.register_region(i + 1, t, sp)
    log = torch.empty(R * (small_bytes + 4096), dtype=torch.uint8, device=dev)
    ctx.log_attach(log)
    res = cc.Result()

    def timed(fn, reps=10):
        ts = []
        for _ in range(reps + 2):
            for t in regs:
                t[::sp * 8] ^= 1
            ctx.log_reset()
            torch.cuda.synchronize()
            t0 = time.perf_counter_ns()
            fn()
            torch.cuda.synchronize()
            ts.append((time.perf_counter_ns() - t0) / 1e3)
        return statistics.median(ts[2:])

    l0 = ctx.kernel_launches()
    t_batch = timed(lambda: ctx.checkpoint_all(1, res))
    l1 = ctx.kernel_launches()
    rb = res.read()
    t_loop = timed(lambda: [ctx.checkpoint_delta(i + 1, 1, res) for i in range(R)])
    l2 = ctx.kernel_launches()
    ctx.shutdown()
    line = base_line(env, len(rows), 0, base, 0.0,
                     "PAPER.md Fig. 7b / L427 analogue (not a BASELINE config): torch device-to-device copy of 4 GiB (GB/s = read + write) "
                     "with no worker (value), next to an idle and next to a busy persistent worker of B CTAs", {"region_MiB": 256, "page_bytes": P,
                                                                                                                "dirty_pages_per_task": n_mut},
                     "u8")
    line["metric"] = METRICS["overlap"]
    line["footprints"] = rows
    line["many_small_regions"] = {"regions": R, "region_MiB": small_bytes >> 20, "page_bytes": sp, "dirty_pages_total": int(rb.n_dirty),
                                  "cc_checkpoint_all_us": round(t_batch, 1), "launches_per_boundary_batched": (l1 - l0 - 12) // 12,
                                  "loop_of_cc_checkpoint_delta_us": round(t_loop, 1), "launches_per_boundary_loop": (l2 - l1 - 12) // 12,
                                  "speedup": round(t_loop / t_batch, 2)}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ reference arm --

def run_reference(args):
    """The oracle, as it stands, on the box's host cores (this tier's reference arm): same bounded sample as cpu_baseline."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    leg = oracle_leg(args.workload, args)
    line = {"impl": "reference", "metric": METRICS.get(args.workload, METRIC), "value": leg["value"], "unit": UNIT,
            "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": round(leg["seconds_per_pass"] * 1e3, 3), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8", "data": "synthetic",
            "config": {"workload": "%s; each step = the oracle on a bounded sample: %s" % (args.workload, leg["sample"])},
            "cpu_baseline": leg,
            "e2e": {"value": leg["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def respawn_under_torchrun(a):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start the N ranks ourselves, exactly as the
    driver would (one process per GPU, rendezvous on 127.0.0.1), and hand back their exit code.  Rank 0 prints the line."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(a.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    a = parse_args()
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(respawn_under_torchrun(a))
    if a.impl == "reference":
        return run_reference(a)
    env = Env()
    if a.workload in KV:
        run_c2(a, env)
    elif a.workload in ("c1", "c3"):
        small_region_workload(a, env, a.workload)
    elif a.workload == "c4-sparse":
        run_c4_sparse(a, env)
    elif a.workload == "c4-full":
        run_c4_full(a, env)
    elif a.workload == "c5a":
        run_c5a(a, env)
    elif a.workload == "c5b":
        run_c5b(a, env)
    elif a.workload == "overlap":
        run_overlap(a, env)
    env.finish()


if __name__ == "__main__":
    main()
