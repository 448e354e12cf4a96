"""Per-config throughput table (SURVEY.md 8d "What is reported per config"; BASELINE.json configs 1-4):

    python -m paper_2606_23521_b200.sweep [--large-gib 64] [--reps 7]

For every configuration it times, with CUDA events on the launch stream and the log in DEVICE memory, the scan
(a1 + a2), the record writer (a3-a5) and the whole checkpoint, and prints region-GB/s, dirty-GB/s and the fraction
of the HBM roofline under the reporting convention bytes = 2 x region + 3 x dirty:
  C1  64 MiB raw bytes, 4 KiB pages, 1 % dirty          (fits L2: reported cold -- 512 MiB written in between -- and warm)
  C2  8 GiB KV cache, 64 KiB blocks, 8,192 dirty
  C3  64 MiB LoRA adapters, 64 KiB pages, 5 % dirty      (cold and warm)
  C4  `--large-gib` GiB bf16 region at 4 / 16 / 64 KiB pages: 0.1 % dirty (scan-bound), and 100 % dirty
      (writer-bound) on the largest slice whose log fits beside region and shadow; for the 100 % case also the fused
      single pass, whose per-page early-out stops reading a page at its first difference.
Inputs come from the seeded generators of synth/ (DESIGN.md section 4).  Prints one JSON object per config.
"""
import argparse
import json
import os
import statistics
import sys

import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import synth  # noqa: E402

from . import binding as cc  # noqa: E402


def _peak():
    try:
        d = json.load(open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")))
        return float(d["hbm_gbs"])
    except Exception:
        return 6650.0


def _time_config(name, cur, P, rearm, k_expect, reps, cold, peak, fused=False, note=None):
    dev = cur.device
    N = cur.numel()
    ctx = cc.Context(dev.index or 0)
    ctx.register_region(1, cur, P)                         # shadow := cur
    n_pages = (N + P - 1) // P
    cap = (n_pages if fused else k_expect) * (16 + P) + 32
    log = torch.empty(cap, dtype=torch.uint8, device=dev)
    ctx.log_attach(log)
    stream = torch.cuda.current_stream()
    scratch = torch.empty(512 << 20, dtype=torch.uint8, device=dev) if cold else None
    res = cc.Result()
    t_scan, t_gather, t_total = [], [], []
    for it in range(reps + 2):
        rearm(it)
        if scratch is not None:
            scratch.fill_(it & 0xFF)                       # push the region out of L2
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        for e in evs:
            e.record(stream)
        torch.cuda.synchronize()
        evs[0].record(stream)
        ctx.trace_events(evs[1], evs[2])
        (ctx.checkpoint_delta_fused if fused else ctx.checkpoint_delta)(1, it, res)
        evs[3].record(stream)
        torch.cuda.synchronize()
        ctx.trace_events(None, None)
        r = res.read()
        assert r.status == 0 and r.n_dirty == k_expect, (name, r.as_dict(), k_expect)
        ctx.log_reset()
        if it >= 2:
            t_scan.append(evs[0].elapsed_time(evs[2]))
            t_gather.append(evs[2].elapsed_time(evs[3]))
            t_total.append(evs[0].elapsed_time(evs[3]))
    ctx.shutdown()
    ts, tg, tt = statistics.median(t_scan), statistics.median(t_gather), statistics.median(t_total)
    kP = k_expect * P
    out = {"config": name, "region_bytes": N, "page_bytes": P, "dirty_pages": k_expect, "l2": "cold" if cold else "as is",
           "path": "fused single pass" if fused else "scan + compact + gather",
           "ms": {"scan_compact": round(ts, 4), "gather_commit_shadow": round(tg, 4), "total": round(tt, 4), "best_total": round(min(t_total), 4)},
           "region_GBps": {"scan": round(N / ts / 1e6, 1), "total": round(N / tt / 1e6, 1)},
           "dirty_GBps": {"writer": round(kP / max(tg, 1e-6) / 1e6, 1), "total": round(kP / tt / 1e6, 1)},
           "hbm_GBps_2N_3kP": round((2 * N + 3 * kP) / tt / 1e6, 1),
           "frac_of_measured_peak": round((2 * N + 3 * kP) / tt / 1e6 / peak, 4),
           "frac_of_8000": round((2 * N + 3 * kP) / tt / 1e6 / 8000, 4)}
    if not fused:
        out["scan_frac_of_measured_peak"] = round(2 * N / ts / 1e6 / peak, 4)
    if note:
        out["note"] = note
    print(json.dumps(out), flush=True)
    del log
    torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--large-gib", type=int, default=64)
    ap.add_argument("--reps", type=int, default=7)
    ap.add_argument("--only", default="")
    a = ap.parse_args()
    dev = torch.device("cuda", 0)
    peak = _peak()
    want = set(a.only.split(",")) if a.only else None

    def on(c):
        return want is None or c in want

    # ---- C1 ----
    if on("c1"):
        cur = synth.raw_region(64 << 20, 1001, dev)
        pages, offs, masks = synth.sparse_xor_flips(cur, 4096, 0.01, 1001)
        synth.toggle_flips(cur, offs, masks)                        # back to the registered state; re-armed per iteration
        for cold, fused in ((True, False), (False, False), (False, True)):
            _time_config("C1 raw 64 MiB / 4 KiB / 1 % dirty", cur, 4096, lambda it: synth.toggle_flips(cur, offs, masks),
                         len(pages), a.reps, cold, peak, fused=fused)
        del cur
    # ---- C2 ----
    if on("c2"):
        layers, blocks, seqs = 32, 4096, 256
        cur = synth.kv_cache_region(layers, blocks, 1002, dev)
        _time_config("C2 KV cache 8 GiB / 64 KiB / 8192 dirty", cur, 65536,
                     lambda it: synth.kv_decode_step(cur, layers, blocks, seqs, 3000 + it), layers * seqs, a.reps, False, peak)
        del cur
    # ---- C3 ----
    if on("c3"):
        cur = synth.lora_region(32, 1003, dev)
        k3 = 52
        for cold, fused in ((True, False), (False, False), (False, True)):
            _time_config("C3 LoRA 64 MiB / 64 KiB / 5 % dirty", cur, 65536, lambda it: synth.lora_update(cur, 65536, 0.05, 4000 + it),
                         k3, a.reps, cold, peak, fused=fused)
        del cur
    torch.cuda.empty_cache()
    # ---- C4 ----
    if on("c4"):
        free, _ = torch.cuda.mem_get_info()
        gib = a.large_gib
        while gib > 1 and 2 * (gib << 30) + (6 << 30) > free:
            gib //= 2
        N = gib << 30
        cur = synth.bf16_normal_region(N, 1004, dev)
        for P in (4096, 16384, 65536):
            pages, offs, masks = synth.sparse_xor_flips(cur, P, 0.001, 1004 + P)
            synth.toggle_flips(cur, offs, masks)
            _time_config("C4 sparse %d GiB / %d KiB / 0.1 %% dirty" % (gib, P >> 10), cur, P,
                         lambda it: synth.toggle_flips(cur, offs, masks), len(pages), a.reps, False, peak,
                         note=None if gib == a.large_gib else "region halved to fit region + shadow in free HBM")
        del cur
        torch.cuda.empty_cache()
        # 100 % dirty: region + shadow + log (3 x N) must fit
        free, _ = torch.cuda.mem_get_info()
        g2 = a.large_gib
        while g2 > 1 and 3 * (g2 << 30) + (g2 << 23) + (6 << 30) > free:
            g2 //= 2
        N = g2 << 30
        cur = synth.bf16_normal_region(N, 1004, dev)
        for P in (4096, 16384, 65536):
            n_pages = N // P
            g = synth.gen(1004 + P, dev)
            offs = torch.arange(n_pages, device=dev) * P + torch.randint(0, P, (n_pages,), generator=g, device=dev)
            masks = torch.randint(1, 256, (n_pages,), generator=g, device=dev, dtype=torch.int64).to(torch.uint8)
            for fused in (False, True):
                _time_config("C4 full %d GiB / %d KiB / 100 %% dirty" % (g2, P >> 10), cur, P,
                             lambda it: synth.toggle_flips(cur, offs, masks), n_pages, max(3, a.reps // 2), False, peak, fused=fused,
                             note="largest power-of-two slice whose log fits beside region and shadow (SURVEY.md 8d fallback ii)")
        del cur


if __name__ == "__main__":
    main()
