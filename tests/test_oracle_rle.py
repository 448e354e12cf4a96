"""Pins for run-length records ("contiguous dirty ranges use run-length encoding"),
-m "not gpu": orc_checkpoint_rle against the pinned orc_checkpoint (run_pages = 1), a pure-Python struct restatement
over every dirty subset of a tiny region, closed forms, and the generalised applier / compactor against the
single-page-record log of the same change."""
import itertools
import struct

import numpy as np
import pytest

import oracle


def _py_crc32c(b: bytes) -> int:
    crc = 0xFFFFFFFF
    for x in b:
        crc ^= x
        for _ in range(8):
            crc = (crc >> 1) ^ 0x82F63B78 if crc & 1 else crc >> 1
    return crc ^ 0xFFFFFFFF


def _py_rle(cur: bytes, P: int, rid: int, epoch: int, dirty, R: int) -> bytes:
    """Group ascending dirty pages into runs that never cross a multiple of R; one record per run."""
    runs = []
    for p in sorted(dirty):
        if runs and runs[-1][-1] + 1 == p and p % R != 0:
            runs[-1].append(p)
        else:
            runs.append([p])
    out = b""
    for run in runs:
        payload = cur[run[0] * P:(run[-1] + 1) * P]
        out += struct.pack("<IIII", rid, run[0], len(payload), _py_crc32c(payload)) + payload
    if runs:
        cp = struct.pack("<QII", epoch, rid, len(runs))
        out += struct.pack("<IIII", 0xFFFFFFFF, 0xFFFFFFFF, 16, _py_crc32c(cp)) + cp
    return out


def _pair(N, P, dirty, seed=0):
    rng = np.random.default_rng(seed)
    cur = rng.integers(0, 256, N, dtype=np.uint8)
    sh = cur.copy()
    for p in dirty:
        sh[p * P + int(rng.integers(0, min(P, N - p * P)))] ^= 0x5A
    return cur, sh


def test_run_pages_1_is_the_plain_checkpoint():
    P, n_pages = 64, 41
    N = P * n_pages - 32
    cur, sh = _pair(N, P, [0, 1, 2, 7, 8, 30, 39, 40])
    a, b = sh.copy(), sh.copy()
    la, lb = np.zeros(4096, np.uint8), np.zeros(4096, np.uint8)
    st1, D1, nb1, W1 = oracle.checkpoint(cur, a, P, 3, 9, la, 16)
    st2, D2, runs, nb2, W2 = oracle.checkpoint_rle(cur, b, P, 3, 9, 1, lb, 16)
    assert (st1, nb1, W1) == (st2, nb2, W2) and runs == len(D1) == 8 and D1.tolist() == D2.tolist()
    assert np.array_equal(la, lb) and np.array_equal(a, b)


@pytest.mark.parametrize("R", [1, 2, 4, 8])
def test_brute_force_every_dirty_subset(R):
    P, n_pages = 16, 6
    N = P * n_pages - 8                                   # short tail page
    base = bytes((11 * i + 3) & 0xFF for i in range(N))
    for dirty in itertools.chain.from_iterable(itertools.combinations(range(n_pages), r) for r in range(n_pages + 1)):
        cur = np.frombuffer(base, np.uint8)
        sh = cur.copy()
        for p in dirty:
            sh[p * P] ^= 1
        exp = _py_rle(base, P, 5, 77, dirty, R)
        log = np.zeros(256, np.uint8)
        st, D, runs, nb, W = oracle.checkpoint_rle(cur, sh, P, 5, 77, R, log, 0)
        assert st == 0 and D.tolist() == list(dirty) and nb == len(exp) == W
        assert log[:nb].tobytes() == exp and not log[nb:].any() and np.array_equal(sh, cur)


def test_closed_forms_and_the_paper_s_contiguous_range():
    P, n_pages, R = 64, 50, 8
    N = P * n_pages
    cur, sh = _pair(N, P, range(n_pages))                 # all dirty: ceil(50/8) = 7 runs
    log = np.zeros(N + 1024, np.uint8)
    st, D, runs, nb, W = oracle.checkpoint_rle(cur, sh, P, 1, 1, R, log, 0)
    assert (st, D.size, runs, nb) == (0, 50, 7, N + 16 * 7 + 32)
    # a contiguous dirty range inside one aligned window is ONE record (L221)
    cur, sh = _pair(N, P, [17, 18, 19, 20, 21])
    log = np.zeros(4096, np.uint8)
    st, D, runs, nb, W = oracle.checkpoint_rle(cur, sh, P, 1, 2, R, log, 0)
    assert (D.tolist(), runs, nb) == ([17, 18, 19, 20, 21], 1, 16 + 5 * P + 32)
    assert log[:16].view(np.uint32).tolist()[:3] == [1, 17, 5 * P]
    # the same range crossing a multiple of R splits there: [22,23] + [24,25]
    cur, sh = _pair(N, P, [22, 23, 24, 25])
    st, D, runs, nb, W = oracle.checkpoint_rle(cur, sh, P, 1, 3, R, np.zeros(4096, np.uint8), 0)
    assert runs == 2 and nb == 2 * 16 + 4 * P + 32
    # log full: nothing written, shadow untouched, a retry gives the identical delta
    cur, sh = _pair(N, P, [3, 4, 9])
    sh0 = sh.copy()
    small = np.zeros(2 * 16 + 3 * P + 32 - 1, np.uint8)
    st, D, runs, nb, W = oracle.checkpoint_rle(cur, sh, P, 1, 4, R, small, 0)
    assert (st, runs, nb, W) == (oracle.ORC_ERR_LOG_FULL, 2, 0, 0) and not small.any() and np.array_equal(sh, sh0)
    # invalid run_pages
    assert oracle.checkpoint_rle(cur, sh, P, 1, 4, 0, small, 0)[0] == oracle.ORC_ERR_INVALID
    assert oracle.checkpoint_rle(cur, sh, P, 1, 4, (1 << 32) // P + 1, small, 0)[0] == oracle.ORC_ERR_INVALID


@pytest.mark.parametrize("R", [2, 4, 16])
def test_applier_and_compactor_treat_a_run_as_its_pages(R):
    P, n_pages = 128, 37
    N = P * n_pages - 48
    dirty = [0, 1, 2, 3, 4, 9, 15, 16, 17, 30, 31, 35, 36]
    cur, old = _pair(N, P, dirty, seed=4)
    la, lb = np.zeros(N + 2048, np.uint8), np.zeros(N + 2048, np.uint8)
    st, D1, nb1, _ = oracle.checkpoint(cur, old.copy(), P, 6, 20, la, 0)
    st, D2, runs, nb2, _ = oracle.checkpoint_rle(cur, old.copy(), P, 6, 20, R, lb, 0)
    assert runs < len(dirty) and nb2 == nb1 - 16 * (len(dirty) - runs)
    # replay: both logs turn the old state into the new one; applied counts records
    t1, t2 = old.copy(), old.copy()
    assert oracle.apply_log(la, nb1, [oracle.Region(6, P, t1)]) == (0, len(dirty), nb1)
    assert oracle.apply_log(lb, nb2, [oracle.Region(6, P, t2)]) == (0, runs, nb2)
    assert np.array_equal(t1, cur) and np.array_equal(t2, cur)
    # a second epoch that rewrites part of a run: last wins page by page
    cur2 = cur.copy()
    cur2[2 * P + 5] ^= 0xFF
    st, D3, runs3, nb3, W3 = oracle.checkpoint_rle(cur2, cur.copy(), P, 6, 21, R, lb, nb2)
    assert runs3 == 1
    t3 = old.copy()
    assert oracle.apply_log(lb, W3, [oracle.Region(6, P, t3)])[0] == 0 and np.array_equal(t3, cur2)
    # compaction of the run log == compaction of the single-page log of the same history
    st, D4, nb4, W4 = oracle.checkpoint(cur2, cur.copy(), P, 6, 21, la, nb1)
    oa, ob = np.zeros(N + 2048, np.uint8), np.zeros(N + 2048, np.uint8)
    ra = oracle.compact_log(la, W4, [oracle.Region(6, P, np.zeros(N, np.uint8))], oa)
    rb = oracle.compact_log(lb, W3, [oracle.Region(6, P, np.zeros(N, np.uint8))], ob)
    assert ra[0] == rb[0] == 0 and ra[1] == rb[1] and ra[3] == rb[3] == len(dirty) and np.array_equal(oa, ob)
    # truncating inside a run record: torn, nothing of that epoch applied
    t4 = old.copy()
    assert oracle.apply_log(lb, 16 + 3 * P, [oracle.Region(6, P, t4)]) == (0, 0, 0) and np.array_equal(t4, old)


def test_applier_rejects_malformed_run_lengths():
    P, n_pages = 32, 8
    N = P * n_pages - 16
    cur = np.arange(N, dtype=np.uint8)

    def one(page, length):
        payload = bytes(length)
        rec = struct.pack("<IIII", 4, page, length, _py_crc32c(payload)) + payload
        cp = struct.pack("<QII", 1, 4, 1)
        log = rec + struct.pack("<IIII", 0xFFFFFFFF, 0xFFFFFFFF, 16, _py_crc32c(cp)) + cp
        t = cur.copy()
        return oracle.apply_log(np.frombuffer(log, np.uint8), len(log), [oracle.Region(4, P, t)]), t

    assert one(2, 3 * P)[0] == (0, 1, 16 + 3 * P + 32)                 # pages 2,3,4
    assert one(6, P + (P - 16))[0][0] == 0                              # pages 6 and the short tail 7
    assert one(7, P - 16)[0][0] == 0                                    # the tail alone
    assert one(2, P + 16)[0][0] == oracle.ORC_ERR_CORRUPT               # ends inside a page
    assert one(6, 2 * P)[0][0] == oracle.ORC_ERR_CORRUPT                # runs past the region's end
    assert one(8, P)[0][0] == oracle.ORC_ERR_CORRUPT                    # page out of range
    assert one(3, 0)[0][0] == oracle.ORC_ERR_CORRUPT                    # empty record
    r, t = one(2, 3 * P)
    assert not t[2 * P:5 * P].any() and np.array_equal(t[:2 * P], cur[:2 * P]) and np.array_equal(t[5 * P:], cur[5 * P:])
