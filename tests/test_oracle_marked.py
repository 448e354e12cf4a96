"""Pins for the allocator-aware checkpoint oracle,
-m "not gpu".  orc_checkpoint_marked / orc_checkpoint_versions are checked against: the already pinned
orc_checkpoint in the two cases where they must coincide with it, a pure-Python struct restatement over every
mark subset of a tiny region, closed-form sizes, the round trip through the pinned applier, and the
consume / log-full / version-advance rules of DESIGN.md readings #29-#32."""
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


def _py_records(cur: bytes, P: int, rid: int, epoch: int, pages) -> bytes:
    out = b""
    for p in pages:
        a = cur[p * P:(p + 1) * P]
        out += struct.pack("<IIII", rid, p, len(a), _py_crc32c(a)) + a
    if pages:
        cp = struct.pack("<QII", epoch, rid, len(pages))
        out += struct.pack("<IIII", 0xFFFFFFFF, 0xFFFFFFFF, 16, _py_crc32c(cp)) + cp
    return out


def _bitmap(n_pages, pages, extra_words=0):
    bm = np.zeros((n_pages + 31) // 32 + extra_words, dtype=np.uint32)
    for p in pages:
        bm[p >> 5] |= np.uint32(1 << (p & 31))
    return bm


def _region(n, seed):
    rng = np.random.default_rng(seed)
    return rng.integers(0, 256, n, dtype=np.uint8)


@pytest.mark.parametrize("P,n_pages,tail", [(16, 7, 0), (64, 40, 48), (256, 70, 16)])
def test_verify_with_every_page_marked_is_the_plain_checkpoint(P, n_pages, tail):
    N = P * (n_pages - 1) + (tail or P)
    cur = _region(N, 1)
    sh = cur.copy()
    rng = np.random.default_rng(2)
    for p in rng.choice(n_pages, n_pages // 3 + 1, replace=False):
        sh[p * P + int(rng.integers(0, min(P, N - p * P)))] ^= 0x21
    sh[N - 1] ^= 1
    sh1, sh2 = sh.copy(), sh.copy()
    log1, log2 = np.zeros(N + 4096, np.uint8), np.zeros(N + 4096, np.uint8)
    st1, D1, nb1, W1 = oracle.checkpoint(cur, sh1, P, 5, 9, log1, 0)
    bm = _bitmap(n_pages, range(n_pages))
    st2, D2, nb2, W2 = oracle.checkpoint_marked(cur, sh2, P, 5, 9, bm, log2, 0, verify=True)
    assert (st1, nb1, W1) == (st2, nb2, W2) and D1.tolist() == D2.tolist() and len(D1) > 1
    assert np.array_equal(log1, log2) and np.array_equal(sh1, sh2) and np.array_equal(sh2, cur)


def test_trusted_marks_equal_to_the_dirty_set_give_the_plain_checkpoint():
    P, n_pages = 64, 33
    N = P * n_pages - 16
    cur = _region(N, 3)
    sh = cur.copy()
    dirty = [0, 5, 31, 32]
    for p in dirty:
        sh[p * P + 3] ^= 0x80
    sh1, sh2 = sh.copy(), sh.copy()
    log1, log2 = np.zeros(4096, np.uint8), np.zeros(4096, np.uint8)
    r1 = oracle.checkpoint(cur, sh1, P, 2, 77, log1, 32)
    r2 = oracle.checkpoint_marked(cur, sh2, P, 2, 77, _bitmap(n_pages, dirty), log2, 32)
    assert r1[0] == r2[0] == 0 and r1[1].tolist() == r2[1].tolist() == dirty and r1[2:] == r2[2:]
    assert np.array_equal(log1, log2) and np.array_equal(sh1, sh2)


def test_brute_force_every_mark_subset_tiny_region():
    P, n_pages = 16, 5
    N = 72                                   # four pages of 16 bytes and a short tail page of 8
    cur = bytes((7 * i + 1) & 0xFF for i in range(N))
    truly_dirty = {1, 4}
    sh0 = bytearray(cur)
    sh0[P + 2] ^= 1
    sh0[N - 1] ^= 0x10
    for marks in itertools.chain.from_iterable(itertools.combinations(range(n_pages), r) for r in range(n_pages + 1)):
        for verify in (False, True):
            exp_pages = [p for p in marks if (not verify or p in truly_dirty)]
            exp = _py_records(cur, P, 3, 11, exp_pages)
            sh = np.frombuffer(bytes(sh0), dtype=np.uint8).copy()
            log = np.zeros(256, np.uint8)
            st, D, nb, W = oracle.checkpoint_marked(np.frombuffer(cur, np.uint8), sh, P, 3, 11,
                                                    _bitmap(n_pages, marks), log, 0, verify=verify)
            assert st == 0 and D.tolist() == exp_pages and nb == len(exp) == W
            assert log[:nb].tobytes() == exp and not log[nb:].any()
            # the shadow is refreshed for exactly the logged pages
            want = bytearray(sh0)
            for p in exp_pages:
                want[p * P:(p + 1) * P] = cur[p * P:(p + 1) * P]
            assert sh.tobytes() == bytes(want)


def test_no_shadow_and_bits_beyond_n_pages_ignored():
    P, n_pages = 32, 10
    cur = _region(P * n_pages, 4)
    bm = _bitmap(n_pages, [2, 9], extra_words=1)
    bm[0] |= np.uint32(1 << 10) | np.uint32(1 << 31)     # pages 10, 31 do not exist
    bm[1] = 0xFFFFFFFF
    log = np.zeros(1024, np.uint8)
    st, D, nb, W = oracle.checkpoint_marked(cur, None, P, 1, 1, bm, log, 0)
    assert st == 0 and D.tolist() == [2, 9] and nb == 2 * (16 + P) + 32
    assert log[:nb].tobytes() == _py_records(cur.tobytes(), P, 1, 1, [2, 9])
    # verify needs a shadow
    assert oracle.checkpoint_marked(cur, None, P, 1, 1, bm, log, 0, verify=True)[0] == oracle.ORC_ERR_INVALID


def test_consume_and_log_full():
    P, n_pages = 64, 12
    cur = _region(P * n_pages, 5)
    sh = cur.copy()
    sh[64 * 3] ^= 1
    sh_before = sh.copy()
    marks = [3, 4, 7]
    need = 3 * (16 + P) + 32
    bm = _bitmap(n_pages, marks)
    log = np.zeros(need - 1, np.uint8)
    st, D, nb, W = oracle.checkpoint_marked(cur, sh, P, 1, 1, bm, log, 0, consume=True)
    assert st == oracle.ORC_ERR_LOG_FULL and D.tolist() == marks and nb == 0 and W == 0
    assert not log.any() and np.array_equal(sh, sh_before) and np.array_equal(bm, _bitmap(n_pages, marks))
    log = np.zeros(need, np.uint8)
    st, D, nb, W = oracle.checkpoint_marked(cur, sh, P, 1, 1, bm, log, 0, consume=True)
    assert st == 0 and nb == need == W and not bm.any() and np.array_equal(sh, cur)
    # consumed bitmap -> nothing to do
    st, D, nb, W = oracle.checkpoint_marked(cur, sh, P, 1, 2, bm, log, W, consume=True)
    assert (st, D.size, nb, W) == (0, 0, 0, need)
    # verify mode, marks on clean pages: empty epoch, marks still consumed
    bm = _bitmap(n_pages, [1, 2])
    st, D, nb, W2 = oracle.checkpoint_marked(cur, sh, P, 1, 3, bm, log, W, verify=True, consume=True)
    assert (st, D.size, nb, W2) == (0, 0, 0, W) and not bm.any()


@pytest.mark.parametrize("verify", [False, True])
def test_round_trip_through_the_applier_when_marks_cover_the_dirty_set(verify):
    P, n_pages = 128, 50
    N = P * n_pages - 32
    old = _region(N, 6)
    cur = old.copy()
    rng = np.random.default_rng(7)
    dirty = sorted(rng.choice(n_pages, 9, replace=False).tolist() + [n_pages - 1])
    dirty = sorted(set(dirty))
    for p in dirty:
        cur[p * P + 1] ^= 0xFF
    marks = sorted(set(dirty) | {0, 13, 14})
    sh = old.copy()
    log = np.zeros(N + 4096, np.uint8)
    st, D, nb, W = oracle.checkpoint_marked(cur, sh, P, 8, 4, _bitmap(n_pages, marks), log, 0, verify=verify)
    assert st == 0 and D.tolist() == (dirty if verify else marks)
    target = old.copy()
    r = oracle.apply_log(log, nb, [oracle.Region(8, P, target)])
    assert r == (0, len(D), nb) and np.array_equal(target, cur) and np.array_equal(sh, cur)


def test_version_counters():
    P, n_pages = 64, 20
    N = P * n_pages - 16
    cur = _region(N, 8)
    ver = np.arange(100, 100 + n_pages, dtype=np.uint64)
    com = ver.copy()
    bumped = [0, 7, 19]
    for p in bumped:
        ver[p] += np.uint64(1 + p)
    log = np.zeros(8192, np.uint8)
    # log full: nothing advances
    small = np.zeros(100, np.uint8)
    com0 = com.copy()
    st, D, nb, W = oracle.checkpoint_versions(cur, None, P, 6, 1, ver, com, small, 0)
    assert st == oracle.ORC_ERR_LOG_FULL and D.tolist() == bumped and np.array_equal(com, com0) and not small.any()
    st, D, nb, W = oracle.checkpoint_versions(cur, None, P, 6, 1, ver, com, log, 0)
    assert st == 0 and D.tolist() == bumped and np.array_equal(com, ver)
    assert nb == 2 * (16 + P) + (16 + P - 16) + 32
    assert log[:nb].tobytes() == _py_records(cur.tobytes(), P, 6, 1, bumped)
    # same bytes as the bitmap form with marks = {version != committed}
    log2 = np.zeros(8192, np.uint8)
    r2 = oracle.checkpoint_marked(cur, None, P, 6, 1, _bitmap(n_pages, bumped), log2, 0)
    assert r2[2] == nb and np.array_equal(log, log2)
    # nothing bumped -> empty
    st, D, nb2, W2 = oracle.checkpoint_versions(cur, None, P, 6, 2, ver, com, log, W)
    assert (st, D.size, nb2, W2) == (0, 0, 0, W)
    # a version that wraps to a smaller value is still "different"
    ver[3] = 0
    sh = cur.copy()
    sh[3 * P] ^= 1
    st, D, nb3, W3 = oracle.checkpoint_versions(cur, sh, P, 6, 3, ver, com, log, W)
    assert st == 0 and D.tolist() == [3] and com[3] == 0 and np.array_equal(sh, cur)
