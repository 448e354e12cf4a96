"""cc_dirty_pages_static -- the dirty list for callers that cannot allocate -- against the regular path.

Some users of this library want "which pages changed since the last commit?" at a moment when device allocation
is off the table: next to a resident persistent kernel (cudaMalloc synchronises the GPU and can wait forever on a
kernel that never exits), inside a server whose memory pool already owns all of HBM, or from a
fault handler that must look before it touches anything.  cc_dirty_pages_static serves them from a fixed 2 MiB
scratch array that lives inside libconcordia.so; the regular path (cc_register_region -> cc_scan_only ->
cc_dirty_list) keeps the same scratch in a caller-allocated workspace.  Both must give the same ascending list,
entry for entry (integer work: exact equality, the bar of every other parity test here).

The scratch array is shared by all calls and remembers the last one, so each case runs the new entry point TWICE
IN A ROW on different dirty sets -- the second one smaller, so that bits left over from the first would show.

This file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a
failure here must not hide the parity tests.  It holds no state of its own and passes alone in a fresh process
as well as after everything else.
"""
import numpy as np
import pytest
import torch

import paper_2606_23521_b200 as cc


def _region(n_bytes, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    return torch.randint(0, 256, (n_bytes,), dtype=torch.uint8, generator=g).cuda()


def _dirty(cur, P, pages, seed):
    """Flip one byte in each of `pages` (first byte, last byte or a seeded one in between)."""
    rng = np.random.default_rng(seed)
    N = cur.numel()
    idx = []
    for j, p in enumerate(pages):
        plen = min(P, N - p * P)
        idx.append(p * P + (0, plen - 1, int(rng.integers(0, plen)))[j % 3])
    idx = torch.tensor(idx, dtype=torch.int64, device=cur.device)
    cur[idx] = cur[idx] ^ 0x5A


def _existing_path(cur, shadow, P):
    ctx = cc.Context()
    ctx.register_region(1, cur, P, shadow=shadow, snapshot_now=False)
    res = cc.Result()
    ctx.scan_only(1, res)
    torch.cuda.synchronize()
    D = ctx.dirty_list(1).tolist()
    assert res.read().n_dirty == len(D)
    ctx.shutdown()
    return D


def _static_path(cur, shadow, P, d_list, d_count):
    d_list.fill_(-1)
    d_count.fill_(-1)
    cc.dirty_pages_static(cur, shadow, P, d_list, d_count)
    torch.cuda.synchronize()
    k = int(d_count.item())
    return k, d_list[:min(k, d_list.numel())].tolist()


# (region bytes, page bytes): several ranking tiles (32,768 pages each) with a ragged last page; the 4 KiB /
# 64 KiB shapes of the benchmarks; a page that is not a whole number of 4 KiB segments
SHAPES = [(100_003 * 256 + 48, 256), (16 << 20, 4096), (24 << 20, 65536), (700 * 4112 + 16, 4112)]


@pytest.mark.gpu
@pytest.mark.parametrize("n_bytes,P", SHAPES)
def test_static_scratch_entry_point_matches_the_workspace_path_twice_in_a_row(n_bytes, P):
    n_pages = (n_bytes + P - 1) // P
    cur = _region(n_bytes, 2301)
    shadow = cur.clone()
    d_list = torch.empty(n_pages, dtype=torch.int32, device="cuda")      # the caller's buffers, made once
    d_count = torch.empty(1, dtype=torch.int32, device="cuda")
    rng = np.random.default_rng(n_pages)

    # first call: ~3 % of the pages + the first and the last (short) page
    pages1 = sorted(set(rng.choice(n_pages, max(2, n_pages * 3 // 100), replace=False).tolist()) | {0, n_pages - 1})
    _dirty(cur, P, pages1, 1)
    want1 = _existing_path(cur, shadow, P)
    assert want1 == pages1                                   # the regular path sees exactly what was flipped
    k1, got1 = _static_path(cur, shadow, P, d_list, d_count)
    assert k1 == len(want1) and got1 == want1

    # second call right after it, on a different and much smaller dirty set: nothing of call 1 may survive
    shadow.copy_(cur)
    pages2 = sorted(set(rng.choice(n_pages, 5, replace=False).tolist()) | {n_pages // 2})
    _dirty(cur, P, pages2, 2)
    want2 = _existing_path(cur, shadow, P)
    k2, got2 = _static_path(cur, shadow, P, d_list, d_count)
    assert k2 == len(want2) and got2 == want2 == pages2

    # and a clean region gives an empty list
    shadow.copy_(cur)
    k3, got3 = _static_path(cur, shadow, P, d_list, d_count)
    assert (k3, got3) == (0, []) and _existing_path(cur, shadow, P) == []


@pytest.mark.gpu
def test_static_scratch_short_list_reports_the_full_count():
    P, n_pages = 4096, 4096
    cur = _region(P * n_pages, 7)
    shadow = cur.clone()
    pages = list(range(3, n_pages, 37))
    _dirty(cur, P, pages, 3)
    d_list = torch.empty(10, dtype=torch.int32, device="cuda")
    d_count = torch.empty(1, dtype=torch.int32, device="cuda")
    k, got = _static_path(cur, shadow, P, d_list, d_count)
    assert k == len(pages) and got == pages[:10]
    # count only
    cc.dirty_pages_static(cur, shadow, P, d_list[:0], d_count)
    torch.cuda.synchronize()
    assert int(d_count.item()) == len(pages)


def test_static_scratch_refuses_more_pages_than_the_built_in_bitmap_holds():
    """Argument checks come before any CUDA call, so this runs without a GPU: one page too many is
    CC_ERR_STATIC_LIMIT, and nothing is launched (the pointers below are never dereferenced)."""
    import ctypes
    lib = cc.load_library()
    err = ctypes.c_int32(-1)
    P = 16
    fake = ctypes.c_void_p(0x10000)
    args = lambda n: (0, fake, fake, n, P, fake, 1, fake, None, ctypes.byref(err))
    assert lib.cc_dirty_pages_static(*args((cc.CC_STATIC_MAX_PAGES + 1) * P)) == cc.CC_ERR_STATIC_LIMIT
    assert err.value == 0
    assert lib.cc_dirty_pages_static(*args(0)) == cc.CC_ERR_INVALID
    assert lib.cc_dirty_pages_static(*args(24)) == cc.CC_ERR_INVALID                    # not a multiple of 16
    assert lib.cc_dirty_pages_static(0, ctypes.c_void_p(0x10008), fake, 4096, P, fake, 1, fake, None, None) == cc.CC_ERR_INVALID
