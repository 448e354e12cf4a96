"""GPU parity: the fused single pass (cc_checkpoint_delta_fused) vs the CPU oracle, bit-exact,
in both of its regimes: records written inline (the worst case fits in the log) and records written by the
gather kernel afterwards (it does not)."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc
from gpu_util import check_checkpoint_parity

pytestmark = pytest.mark.gpu

SHAPES = [(16, 7, 0), (64, 300, 48), (256, 1033, 0), (4096, 700, 0), (4096, 1337, 1024), (4112, 129, 16),
          (16384, 190, 4096 + 16), (65536, 37, 0), (65536, 21, 65520), (81920, 14, 4096), (1 << 20, 3, 0),
          (3 << 19, 3, 1 << 19)]


def _mutated(P, n_pages, tail, density=3):
    N = (n_pages - 1) * P + (tail or P)
    cur = synth.raw_region(N, 100 + P % 97 + n_pages, "cuda")
    sh = cur.clone()
    rng = np.random.default_rng(P + n_pages)
    for p in sorted(set(rng.integers(0, n_pages, max(1, n_pages // density)).tolist()) | {0, n_pages - 1}):
        plen = min(P, N - p * P)
        sh[p * P + int(rng.integers(0, plen))] ^= 1 << int(rng.integers(0, 8))
    return cur, sh, N


@pytest.mark.parametrize("P,n_pages,tail", SHAPES)
@pytest.mark.parametrize("inline", [True, False])
def test_fused_small_shapes(P, n_pages, tail, inline):
    cur, sh, N = _mutated(P, n_pages, tail)
    n_dirty = int(oracle.scan(cur.cpu().numpy(), sh.cpu().numpy(), P).sum())
    worst = n_pages * (16 + P) + 32
    cap = worst + 64 if inline else n_dirty * (16 + P) + 32      # exact fit: only the gather kernel can be used
    check_checkpoint_parity(cur, sh, P, log_capacity=cap, fused=True, pinned_log=(n_pages % 2 == 1))


def test_fused_empty_all_dirty_and_log_full():
    P, n_pages = 4096, 515
    N = P * n_pages - 2048
    cur = synth.raw_region(N, 7, "cuda")
    ctx, glog, r, olog, nb = check_checkpoint_parity(cur, cur.clone(), P, fused=True)
    assert r.n_dirty == 0 and r.bytes == 0 and not glog.any()
    ctx.shutdown()
    ctx, glog, r, olog, nb = check_checkpoint_parity(cur, ~cur, P, fused=True)
    assert r.n_dirty == n_pages
    ctx.shutdown()
    # one byte short of the need: LOG_FULL, nothing written, shadow untouched (helper compares all of it)
    sh = cur.clone()
    sh[5 * P] ^= 1
    sh[N - 1] ^= 1
    need = 2 * 16 + P + (P - 2048) + 32
    ctx, glog, r, olog, nb = check_checkpoint_parity(cur, sh, P, log_capacity=need - 1, fused=True)
    assert r.status == cc.CC_ERR_LOG_FULL and r.n_dirty == 2 and not glog.any()
    ctx.shutdown()


def test_fused_chains_with_the_other_paths_and_switches_regime_as_the_log_fills():
    """Epochs written alternately by the fused pass, the three-kernel path and the allocator-aware path land back
    to back; the fused pass goes inline while the worst case still fits and falls back to the gather after."""
    P, n_pages = 4096, 256
    cur = synth.raw_region(P * n_pages, 11, "cuda")
    ctx = cc.Context()
    sh = ctx.register_region(1, cur, P)
    worst = n_pages * (16 + P) + 32
    cap = worst + 5 * (3 * (16 + P) + 32)
    log = torch.zeros(cap, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    host_cur = cur.cpu().numpy().copy()
    host_sh = host_cur.copy()
    olog = np.zeros(cap, dtype=np.uint8)
    W = 0
    rng = np.random.default_rng(3)
    res = cc.Result()
    gm = torch.zeros(n_pages // 32, dtype=torch.int32, device="cuda")
    for e in range(12):
        pages = sorted(set(rng.integers(0, n_pages, 3).tolist()))
        for p in pages:
            off = p * P + int(rng.integers(0, P))
            host_cur[off] ^= 0x41
            cur[off] ^= 0x41
        res.clear()
        if e % 3 == 2:
            bm = np.zeros(n_pages // 32, dtype=np.uint32)
            for p in pages:
                bm[p >> 5] |= np.uint32(1 << (p & 31))
            gm.copy_(torch.from_numpy(bm.view(np.int32)))
            ctx.checkpoint_marked(1, e, gm, cc.CC_MARK_VERIFY, res)
        elif e % 3 == 1:
            ctx.checkpoint_delta(1, e, res)
        else:
            ctx.checkpoint_delta_fused(1, e, res)
        torch.cuda.synchronize()
        st, D, nb, W = oracle.checkpoint(host_cur, host_sh, P, 1, e, olog, W)
        r = res.read()
        assert (r.status, r.n_dirty, r.bytes, r.log_offset_after) == (st, D.size, nb, W), (e, r.as_dict())
        assert ctx.dirty_list(1).tolist() == D.tolist()
    assert W > cap - worst          # the later fused epochs ran in the fall-back regime
    assert np.array_equal(log.cpu().numpy(), olog) and np.array_equal(sh.cpu().numpy(), host_sh)
    ctx.shutdown()


@pytest.mark.parametrize("cfg", ["c1", "c3"])
def test_fused_configs_full_size(cfg):
    if cfg == "c1":
        P = 4096
        cur = synth.raw_region(64 << 20, 1001, "cuda")
        sh = cur.clone()
        synth.mutate_byte_flips(cur, P, 0.01, 1001)
    else:
        P = 65536
        cur = synth.lora_region(32, 1003, "cuda")
        sh = cur.clone()
        synth.lora_update(cur, P, 0.05, 1003)
    ctx, glog, r, olog, nb = check_checkpoint_parity(cur, sh, P, fused=True, pinned_log=True)
    assert r.n_dirty == (164 if cfg == "c1" else 52)
    ctx.shutdown()


def test_fused_c2_full_8gib_equals_three_kernel_path():
    free, _ = torch.cuda.mem_get_info()
    if free < 30 * 2**30:
        pytest.skip("needs 30 GiB of device memory")
    layers, blocks, seqs, P = 32, 4096, 256, 65536
    cur = synth.kv_cache_region(layers, blocks, 1002, "cuda")
    ctx = cc.Context()
    sh = ctx.register_region(1, cur, P)
    pages = synth.kv_decode_step(cur, layers, blocks, seqs, 1002)
    k = pages.numel()
    n_pages = layers * blocks
    worst = n_pages * (16 + P) + 32
    log_f = torch.zeros(worst, dtype=torch.uint8, device="cuda")       # inline regime
    need = k * (16 + P) + 32
    log_c = torch.zeros(need, dtype=torch.uint8, device="cuda")
    sh0 = sh.clone()
    res = cc.Result()
    ctx.log_attach(log_f)
    ctx.checkpoint_delta_fused(1, 5, res)
    torch.cuda.synchronize()
    r = res.read()
    assert (r.status, r.n_dirty, r.bytes) == (0, k, need)
    assert ctx.dirty_list(1).tolist() == pages.tolist() and torch.equal(sh, cur)
    sh.copy_(sh0)
    ctx.log_attach(log_c)
    res.clear()
    ctx.checkpoint_delta(1, 5, res)
    torch.cuda.synchronize()
    assert res.read().n_dirty == k
    assert torch.equal(log_f[:need], log_c) and not log_f[need:].any()
    for i in np.random.default_rng(1).integers(0, k, 16).tolist():
        rec = log_f[i * (16 + P):(i + 1) * (16 + P)].cpu().numpy()
        p = int(pages[i])
        page = cur[p * P:(p + 1) * P].cpu().numpy()
        assert rec[:16].view(np.uint32).tolist() == [1, p, P, oracle.crc32c(page)] and np.array_equal(rec[16:], page)
    # fall-back regime (exact-fit log) gives the same bytes
    sh.copy_(sh0)
    log_c.zero_()
    ctx.log_reset()
    res.clear()
    ctx.checkpoint_delta_fused(1, 5, res)
    torch.cuda.synchronize()
    assert res.read().bytes == need and torch.equal(log_f[:need], log_c)
    ctx.shutdown()
