"""Pins for the base-snapshot and log-compactor oracle,
-m "not gpu": coincidence with already pinned functions, a pure-Python dict/struct restatement on random tiny
logs, replay equivalence through the pinned applier, idempotence, identity on already-compact logs, the
truncation sweep, corrupt / log-full behaviour, and the second worked example of SURVEY.md 8c (tests/golden/)."""
import os
import struct

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


def _hex_fixture(name):
    data = bytearray()
    for line in open(os.path.join(HERE, "golden", name)):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        data += bytes(int(x, 16) for x in line.split())
    return bytes(data)


def _py_crc32c(b: bytes) -> int:
    crc = 0xFFFFFFFF
    for x in b:
        crc ^= x
        for _ in range(8):
            crc = (crc >> 1) ^ 0x82F63B78 if crc & 1 else crc >> 1
    return crc ^ 0xFFFFFFFF


def _py_commit(epoch, rid, k):
    cp = struct.pack("<QII", epoch, rid, k)
    return struct.pack("<IIII", 0xFFFFFFFF, 0xFFFFFFFF, 16, _py_crc32c(cp)) + cp


def _py_compact(log: bytes):
    """Restatement for VALID, untorn logs: dict of the last payload per (region, page) + last epoch per region."""
    off, pend, last, last_epoch = 0, [], {}, {}
    while off < len(log):
        rid, pidx, ln, crc = struct.unpack_from("<IIII", log, off)
        if rid == 0xFFFFFFFF:
            epoch, c_rid, k = struct.unpack_from("<QII", log, off + 16)
            assert k == len(pend)
            for (r, p, rec) in pend:
                last[(r, p)] = rec
                last_epoch[r] = epoch
            pend = []
            off += 32
        else:
            pend.append((rid, pidx, log[off:off + 16 + ln]))
            off += 16 + ln
    out = b""
    for r in sorted({r for r, _ in last}):
        pages = sorted(p for rr, p in last if rr == r)
        out += b"".join(last[(r, p)] for p in pages) + _py_commit(last_epoch[r], r, len(pages))
    return out, len(last)


def _random_log(seed, regions, n_epochs, max_k):
    """regions: list of (rid, P, N).  Returns log bytes (numpy)."""
    rng = np.random.default_rng(seed)
    cap = sum((16 + P) * max_k + 32 for _, P, _ in regions) * n_epochs + 64
    log = np.zeros(cap, np.uint8)
    W = 0
    for e in range(n_epochs):
        rid, P, N = regions[int(rng.integers(0, len(regions)))]
        n_pages = (N + P - 1) // P
        k = int(rng.integers(0, min(max_k, n_pages) + 1))
        pages = np.sort(rng.choice(n_pages, k, replace=False)).astype(np.uint32)
        lens = [min(P, N - int(p) * P) for p in pages]
        payloads = rng.integers(0, 256, sum(lens), dtype=np.uint8)
        if k == 0:
            continue           # orc_write_epoch with k = 0 would write a bare commit; exercised separately
        st, W = oracle.write_epoch(log, W, rid, 100 + e, N, P, pages, payloads)
        assert st == 0
    return log[:W].copy()


REGIONS = [(7, 16, 16 * 9 - 8), (2, 32, 32 * 5), (40, 64, 64 * 4 - 16)]


def _oregions(seed=0):
    rng = np.random.default_rng(seed)
    return [oracle.Region(rid, P, rng.integers(0, 256, N, dtype=np.uint8)) for rid, P, N in REGIONS]


def test_snapshot_is_the_all_pages_epoch():
    P, n_pages = 64, 13
    N = P * n_pages - 16
    rng = np.random.default_rng(1)
    cur = rng.integers(0, 256, N, dtype=np.uint8)
    sh = rng.integers(0, 256, N, dtype=np.uint8)
    log = np.zeros(N + 1024, np.uint8)
    st, k, nb, W = oracle.snapshot(cur, sh, P, 9, 3, log, 0)
    assert (st, k, nb, W) == (0, n_pages, (n_pages - 1) * (16 + P) + (16 + P - 16) + 32, nb)
    assert np.array_equal(sh, cur)
    # == the plain checkpoint against a shadow that differs everywhere, and == trusted marks on every page
    log2, log3 = np.zeros_like(log), np.zeros_like(log)
    assert oracle.checkpoint(cur, (~cur).copy(), P, 9, 3, log2, 0)[0] == 0
    bm = np.full((n_pages + 31) // 32, 0xFFFFFFFF, dtype=np.uint32)
    assert oracle.checkpoint_marked(cur, None, P, 9, 3, bm, log3, 0)[0] == 0
    assert np.array_equal(log, log2) and np.array_equal(log, log3)
    # payloads concatenated == the region (north_star "all pages dirty give a full copy")
    g = log[:nb]
    pay = np.concatenate([g[i * (16 + P) + 16: i * (16 + P) + 16 + min(P, N - i * P)] for i in range(n_pages)])
    assert np.array_equal(pay, cur)
    # restoring an empty replacement region from the base snapshot alone
    target = np.zeros(N, np.uint8)
    assert oracle.apply_log(log, nb, [oracle.Region(9, P, target)]) == (0, n_pages, nb) and np.array_equal(target, cur)
    # log full: nothing written, shadow untouched
    sh2 = np.zeros(N, np.uint8)
    small = np.zeros(nb - 1, np.uint8)
    st, k, nb2, W2 = oracle.snapshot(cur, sh2, P, 9, 3, small, 0)
    assert (st, nb2, W2) == (oracle.ORC_ERR_LOG_FULL, 0, 0) and not small.any() and not sh2.any()


@pytest.mark.parametrize("seed", range(12))
def test_compact_matches_python_restatement_and_replays_identically(seed):
    log = _random_log(seed, REGIONS, n_epochs=9, max_k=4)
    exp, n_exp = _py_compact(log.tobytes())
    out = np.zeros(len(log) + 64, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(log, log.size, _oregions(), out)
    assert (st, nb, consumed, n_out) == (0, len(exp), log.size, n_exp)
    assert out[:nb].tobytes() == exp and not out[nb:].any()
    assert nb <= log.size
    # replay equivalence on an arbitrary starting state, every region
    a, b = _oregions(seed + 100), _oregions(seed + 100)
    ra = oracle.apply_log(log, log.size, a)
    rb = oracle.apply_log(out, nb, b)
    assert ra[0] == rb[0] == 0 and rb[1] == n_out and rb[2] == nb
    for x, y in zip(a, b):
        assert np.array_equal(x.base, y.base)
    # idempotent
    out2 = np.zeros_like(out)
    st2, nb2, consumed2, n_out2 = oracle.compact_log(out, nb, _oregions(), out2)
    assert (st2, nb2, consumed2, n_out2) == (0, nb, nb, n_out) and np.array_equal(out, out2)


def test_compact_identity_on_an_already_compact_log_and_empty_inputs():
    # one epoch per region, regions ascending, pages ascending, no duplicates -> unchanged
    log = np.zeros(4096, np.uint8)
    W = 0
    rng = np.random.default_rng(5)
    for rid, P, N in sorted(REGIONS):
        pages = np.array([0, 2, (N + P - 1) // P - 1], dtype=np.uint32)
        lens = [min(P, N - int(p) * P) for p in pages]
        st, W = oracle.write_epoch(log, W, rid, 50 + rid, N, P, pages, rng.integers(0, 256, sum(lens), dtype=np.uint8))
    out = np.zeros(4096, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(log, W, _oregions(), out)
    assert (st, nb, consumed, n_out) == (0, W, W, 9) and np.array_equal(out, log)
    # empty log, and a log of empty epochs only: nothing out
    assert oracle.compact_log(log, 0, _oregions(), out)[:2] == (0, 0)
    empty = np.frombuffer(_py_commit(1, 7, 0) + _py_commit(2, 2, 0), np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(empty, empty.size, _oregions(), np.zeros(64, np.uint8))
    assert (st, nb, consumed, n_out) == (0, 0, 64, 0)


def test_compact_truncation_sweep_corruption_and_capacity():
    log = _random_log(3, REGIONS, n_epochs=5, max_k=3)
    # epoch boundaries of the input
    bounds, off = [0], 0
    raw = log.tobytes()
    while off < len(raw):
        rid, _, ln, _ = struct.unpack_from("<IIII", raw, off)
        off += 16 + ln
        if rid == 0xFFFFFFFF:
            bounds.append(off)
    for t in range(0, len(raw) + 1, 7):
        whole = max(b for b in bounds if b <= t)
        exp, n_exp = _py_compact(raw[:whole])
        out = np.zeros(len(raw) + 64, np.uint8)
        st, nb, consumed, n_out = oracle.compact_log(log, t, _oregions(), out)
        assert (st, nb, consumed, n_out) == (0, len(exp), whole, n_exp) and out[:nb].tobytes() == exp
    # one flipped payload bit anywhere in a committed epoch: CORRUPT and nothing written
    bad = log.copy()
    bad[20] ^= 0x04
    out = np.zeros(len(raw) + 64, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(bad, bad.size, _oregions(), out)
    assert (st, nb, n_out) == (oracle.ORC_ERR_CORRUPT, 0, 0) and not out.any()
    # output one byte too small: LOG_FULL and nothing written
    exp, _ = _py_compact(raw)
    out = np.zeros(len(exp) - 1, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(log, log.size, _oregions(), out)
    assert (st, nb, n_out) == (oracle.ORC_ERR_LOG_FULL, 0, 0) and not out.any()
    out = np.zeros(len(exp), np.uint8)
    assert oracle.compact_log(log, log.size, _oregions(), out)[0] == 0 and out.tobytes() == exp


def test_compact_worked_example_2():
    """SURVEY.md 8c second worked example (224 bytes: epoch 10 = pages 0,1,2 of region 2, epoch 11 = page 2 again).
    Compaction keeps pages 0 and 1 from epoch 10 and page 2 from epoch 11, under one commit for epoch 11."""
    g = _hex_fixture("worked_example_2.txt")
    if len(g) == 64:        # the fixture stores only the epoch-11 tail printed in the survey; rebuild epoch 10
        cur = bytes((3 * i) % 256 for i in range(80))
        e10 = b"".join(struct.pack("<IIII", 2, p, len(cur[p * 32:(p + 1) * 32]), _py_crc32c(cur[p * 32:(p + 1) * 32])) +
                       cur[p * 32:(p + 1) * 32] for p in range(3)) + _py_commit(10, 2, 3)
        g = e10 + g
    assert len(g) == 224 and _py_crc32c(g) == 0x241E68BB          # the survey's one-number check of the whole log
    exp = g[0:48] + g[48:96] + g[160:192] + _py_commit(11, 2, 3)
    out = np.zeros(256, np.uint8)
    region = oracle.Region(2, 32, np.zeros(80, np.uint8))
    st, nb, consumed, n_out = oracle.compact_log(np.frombuffer(g, np.uint8), 224, [region], out)
    assert (st, nb, consumed, n_out) == (0, 160, 224, 3) and out[:160].tobytes() == exp
