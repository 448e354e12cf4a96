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
