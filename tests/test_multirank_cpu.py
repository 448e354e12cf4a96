"""-m "not gpu": the N>1 host logic with world_size 2 over gloo (no GPU, no data-path collective)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import numpy as np
    import oracle
    import synth
    from paper_2606_23521_b200 import sharding
    out = {}
    # every rank owns its own region (different seed) and its own log; same epoch id on all ranks
    seed = sharding.rank_seed(1002, rank)
    cur = synth.kv_cache_region(1, 32, seed, "cpu")
    old = cur.clone()
    pages = synth.kv_decode_step(cur, 1, 32, 4 + rank, seed)
    epoch = sharding.agree_epoch(41)
    log = np.zeros(len(pages) * (16 + 65536) + 32, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur.numpy(), old.numpy().copy(), 65536, 1, epoch, log, 0)
    out["k"] = int(D.size)
    out["seed"] = seed
    # throughput aggregation: sum of units over max of times
    val, mx = sharding.job_throughput(float(cur.numel()), 10.0 * (rank + 1))
    out["val"], out["max_ms"] = val, mx
    # disagreement on the epoch is detected on every rank
    try:
        sharding.agree_epoch(100 + rank)
        out["mismatch"] = False
    except RuntimeError:
        out["mismatch"] = True
    q.put((rank, out))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_without_exchange():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0]["seed"] != res[1]["seed"]
    assert (res[0]["k"], res[1]["k"]) == (4, 5)                  # independent dirty sets per rank
    n = 32 * 65536
    for r in (0, 1):
        assert res[r]["max_ms"] == 20.0
        assert res[r]["val"] == pytest.approx(2 * n / 20e-3)
        assert res[r]["mismatch"] is True


def test_bench_gpus_2_spawns_its_own_ranks_reference_arm():
    """`python bench.py --impl reference --gpus 2` with no torchrun environment re-executes itself under
    torch.distributed.run (two processes, rendezvous on 127.0.0.1): rank 0 alone times the oracle and prints ONE JSON
    line with n_gpus = 2, rank 1 exits 0 without work.  Runs on CPU (the reference arm is the oracle)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    p = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--workload", "c2-small", "--steps", "1", "--warmup", "0"],
                       cwd=root, env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, p.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
