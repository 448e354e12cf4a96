"""Pins for the multi-region boundary oracle, -m "not gpu":
orc_checkpoint_all must be exactly a sequence of the already pinned orc_checkpoint calls in ascending region id."""
import numpy as np

import oracle


def _mk(seed):
    rng = np.random.default_rng(seed)
    specs = [(9, 64, 64 * 7 - 16), (2, 16, 16 * 12), (5, 32, 32 * 9), (7, 128, 128 * 3)]     # ids deliberately unsorted
    regs = []
    for rid, P, N in specs:
        cur = rng.integers(0, 256, N, dtype=np.uint8)
        sh = cur.copy()
        n_pages = (N + P - 1) // P
        for p in rng.choice(n_pages, max(1, n_pages // 3), replace=False):
            sh[p * P + int(rng.integers(0, min(P, N - p * P)))] ^= 0x3C
        regs.append(oracle.Region(rid, P, cur, sh))
    regs[3].shadow = None            # region 7: allocator-aware / immutable, takes no part
    return regs


def _loop(regs, epoch, log, W):
    ks, sts, first = {}, {}, 0
    for r in sorted(regs, key=lambda r: r.region_id):
        if r.shadow is None:
            continue
        st, D, nb, W = oracle.checkpoint(r.base, r.shadow, r.page_bytes, r.region_id, epoch, log, W)
        ks[r.region_id], sts[r.region_id] = D.size, st
        if st and not first:
            first = st
    return first, ks, sts, W


def test_checkpoint_all_is_the_ascending_sequence_of_checkpoints():
    a, b = _mk(1), _mk(1)
    la, lb = np.zeros(4096, np.uint8), np.zeros(4096, np.uint8)
    st, ks, sts, kt, bt, W = oracle.checkpoint_all(a, 12, la, 48)
    first, ks2, sts2, W2 = _loop(b, 12, lb, 48)
    assert st == first == 0 and W == W2 and bt == W - 48 and kt == sum(ks2.values()) > 0
    assert [ks[i] for i, r in enumerate(a) if r.shadow is not None] == [ks2[r.region_id] for r in a if r.shadow is not None]
    assert ks[3] == 0 and sts[3] == 0
    assert np.array_equal(la, lb)
    for x, y in zip(a, b):
        if x.shadow is not None:
            assert np.array_equal(x.shadow, y.shadow) and np.array_equal(x.shadow, x.base)
    # the log's first record belongs to the LOWEST region id (2), not to the first in the list (9)
    assert int(la[48:52].view(np.uint32)[0]) == 2
    # nothing changed since: empty boundary
    st, ks, sts, kt, bt, W3 = oracle.checkpoint_all(a, 13, la, W)
    assert (st, kt, bt, W3) == (0, 0, 0, W)


def test_checkpoint_all_skips_a_region_that_does_not_fit_and_tries_the_rest():
    a, b = _mk(2), _mk(2)
    # capacity: region 2 fits, region 5 does not (one byte short), region 9 is tried afterwards
    st0, D2, nb2, W2 = oracle.checkpoint(b[1].base, b[1].shadow.copy(), 16, 2, 1, np.zeros(8192, np.uint8), 0)
    st0, D5, nb5, _ = oracle.checkpoint(b[2].base, b[2].shadow.copy(), 32, 5, 1, np.zeros(8192, np.uint8), 0)
    cap = nb2 + nb5 - 1
    la = np.zeros(cap, np.uint8)
    lb = np.zeros(cap, np.uint8)
    st, ks, sts, kt, bt, W = oracle.checkpoint_all(a, 1, la, 0)
    first, ks2, sts2, Wb = _loop(b, 1, lb, 0)
    assert st == first == oracle.ORC_ERR_LOG_FULL and W == Wb and np.array_equal(la, lb)
    assert sts[2] == oracle.ORC_ERR_LOG_FULL and sts[1] == 0
    assert not np.array_equal(a[2].shadow, a[2].base)          # region 5 untouched: retry later gives the same delta
    assert np.array_equal(a[1].shadow, a[1].base)
    assert sts[0] == sts2[9] and np.array_equal(a[0].shadow, b[0].shadow)
