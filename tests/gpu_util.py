"""Shared helpers of the GPU parity tests: run the CUDA path and the oracle on the same bytes."""
import numpy as np
import torch

import oracle
import paper_2606_23521_b200 as cc


def gpu_checkpoint(ctx, region_id, epoch, res=None, fused=False):
    res = res or cc.Result()
    res.clear()
    (ctx.checkpoint_delta_fused if fused else ctx.checkpoint_delta)(region_id, epoch, res)
    torch.cuda.synchronize()
    return res.read()


def check_checkpoint_parity(cur: torch.Tensor, shadow0: torch.Tensor, P: int, region_id=3, epoch=17,
                            log_capacity=None, pinned_log=False, W0_epochs=0, fused=False):
    """cur, shadow0: uint8 CUDA tensors.  Runs one checkpoint on GPU and oracle; compares dirty list,
    log bytes, shadow, result fields.  Returns (ctx, log tensor, result, oracle log numpy, nbytes)."""
    N = cur.numel()
    n_pages = (N + P - 1) // P
    cap = log_capacity if log_capacity is not None else n_pages * (16 + P) + 32 + 64
    cur_h = cur.cpu().numpy()
    sh_h = shadow0.cpu().numpy().copy()
    olog = np.zeros(cap, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur_h, sh_h, P, region_id, epoch, olog, 0)

    ctx = cc.Context()
    shadow = shadow0.clone()
    ctx.register_region(region_id, cur, P, shadow=shadow, snapshot_now=False)
    if pinned_log:
        glog = torch.zeros(cap, dtype=torch.uint8, pin_memory=True)
    else:
        glog = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(glog, committed)
    r = gpu_checkpoint(ctx, region_id, epoch, fused=fused)
    assert r.seq_done == 1
    assert r.status == st, (r.status, st)
    assert r.n_dirty == D.size, (r.n_dirty, D.size)
    assert ctx.dirty_list(region_id).tolist() == D.tolist()
    assert r.bytes == nb and r.log_offset_after == W
    assert int(committed.item()) == W
    assert r.epoch == epoch
    g = glog.cpu().numpy()
    assert np.array_equal(g, olog), "log bytes differ at %s" % np.nonzero(g != olog)[0][:8]
    assert np.array_equal(shadow.cpu().numpy(), sh_h), "shadow differs"
    assert np.array_equal(cur.cpu().numpy(), cur_h), "live region was modified"
    return ctx, glog, r, olog, nb


def verify_all_dirty(cur, log, offs, masks, P, region_id, epoch, chunk=1 << 30, threads=16, log_is_host=False):
    """Every record of an all-dirty checkpoint (one seeded flip per page: synth.all_dirty_flips) against oracle.checkpoint,
    1 GiB chunk by chunk (oracle/chunked.py).  cur: the live region AFTER the flips; the shadow the checkpoint started
    from is cur with the flips undone.  Returns (k, log bytes, D) as the oracle sees them; raises on the first mismatch."""
    from oracle import chunked
    N = cur.numel()
    o_cpu, m_cpu = offs.cpu().numpy(), masks.cpu().numpy()

    def fetch_shadow0(o, n):
        a = cur[o:o + n].cpu().numpy()
        lo, hi = (o // P), ((o + n) // P)                          # one flip per page, ascending
        a[o_cpu[lo:hi] - o] ^= m_cpu[lo:hi]
        return a
    fl = (lambda o, n: log[o:o + n].numpy()) if log_is_host else (lambda o, n: log[o:o + n].cpu().numpy())
    return chunked.verify_checkpoint_chunked(N, P, region_id, epoch, lambda o, n: cur[o:o + n].cpu().numpy(), fetch_shadow0, fl,
                                             chunk_bytes=chunk, threads=threads)
