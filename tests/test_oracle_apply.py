"""Pins for the apply oracle (-m "not gpu"): round trip, idempotence, truncation, corruption."""
import struct

import numpy as np
import pytest

import oracle
import synth


def _two_epoch_log(P=64, n_pages=12, tail=32):
    """old snapshot, two checkpoints (second rewrites one page of the first), returns pieces."""
    N = (n_pages - 1) * P + tail
    rng = np.random.default_rng(5)
    old = rng.integers(0, 256, N, dtype=np.uint8)
    cur = old.copy()
    sh = old.copy()
    log = np.zeros(4096, dtype=np.uint8)
    for p in (1, 4, n_pages - 1):
        cur[p * P + 3] ^= 0x55
    st, D1, nb1, W = oracle.checkpoint(cur, sh, P, 3, 100, log, 0)
    mid = cur.copy()
    for p in (4, 7):
        cur[p * P + 9] ^= 0xAA
    st, D2, nb2, W = oracle.checkpoint(cur, sh, P, 3, 101, log, W)
    return old, mid, cur, log, nb1, nb2, P


def test_round_trip_and_idempotence():
    old, mid, cur, log, nb1, nb2, P = _two_epoch_log()
    reg, sh = old.copy(), old.copy()
    r = [oracle.Region(3, P, reg, sh)]
    assert oracle.apply_log(log, nb1 + nb2, r) == (0, 5, nb1 + nb2)
    assert (reg == cur).all() and (sh == cur).all()
    assert oracle.apply_log(log, nb1 + nb2, r) == (0, 5, nb1 + nb2)      # idempotent
    assert (reg == cur).all()
    # apply-then-checkpoint -> empty (apply refreshes the shadow, reading #18)
    l2 = np.zeros(64, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(reg, sh, P, 3, 102, l2, 0)
    assert D.size == 0 and nb == 0


def test_truncation_sweep_every_byte():
    """For every cut t the result equals applying the largest whole-epoch prefix <= t, status OK."""
    old, mid, cur, log, nb1, nb2, P = _two_epoch_log()
    total = nb1 + nb2
    for t in range(total + 1):
        reg = old.copy()
        st, applied, consumed = oracle.apply_log(log, t, [oracle.Region(3, P, reg)])
        assert st == 0
        if t < nb1:
            assert (applied, consumed) == (0, 0) and (reg == old).all()
        elif t < total:
            assert (applied, consumed) == (3, nb1) and (reg == mid).all()
        else:
            assert (applied, consumed) == (5, total) and (reg == cur).all()


def test_one_bit_payload_corruption():
    old, mid, cur, log, nb1, nb2, P = _two_epoch_log()
    total = nb1 + nb2
    # flip a payload bit in the first record of epoch 2 -> CORRUPT, epoch 1 applied, epoch 2 not
    bad = log.copy()
    bad[nb1 + 16 + 5] ^= 0x04
    reg = old.copy()
    assert oracle.apply_log(bad, total, [oracle.Region(3, P, reg)]) == (oracle.ORC_ERR_CORRUPT, 3, nb1)
    assert (reg == mid).all()
    # flip a payload bit in epoch 1 -> nothing applied
    bad = log.copy()
    bad[16 + 0] ^= 0x80
    reg = old.copy()
    assert oracle.apply_log(bad, total, [oracle.Region(3, P, reg)]) == (oracle.ORC_ERR_CORRUPT, 0, 0)
    assert (reg == old).all()


@pytest.mark.parametrize("field,value", [("region", 99), ("page", 10_000), ("len", 48), ("crc", 0xDEADBEEF)])
def test_bad_header_fields(field, value):
    old, mid, cur, log, nb1, nb2, P = _two_epoch_log()
    bad = log.copy()
    off = nb1   # first header of epoch 2
    idx = {"region": 0, "page": 4, "len": 8, "crc": 12}[field]
    bad[off + idx: off + idx + 4] = np.frombuffer(struct.pack("<I", value), dtype=np.uint8)
    reg = old.copy()
    st, applied, consumed = oracle.apply_log(bad, nb1 + nb2, [oracle.Region(3, P, reg)])
    assert (st, applied, consumed) == (oracle.ORC_ERR_CORRUPT, 3, nb1) and (reg == mid).all()


def test_len_larger_than_remaining_is_torn_not_corrupt():
    old, mid, cur, log, nb1, nb2, P = _two_epoch_log()
    bad = log.copy()
    bad[nb1 + 8: nb1 + 12] = np.frombuffer(struct.pack("<I", 1 << 30), dtype=np.uint8)
    reg = old.copy()
    assert oracle.apply_log(bad, nb1 + nb2, [oracle.Region(3, P, reg)]) == (0, 3, nb1)


@pytest.mark.parametrize("what", ["k", "region", "crc", "pageidx", "len"])
def test_bad_commit_record(what):
    old, mid, cur, log, nb1, nb2, P = _two_epoch_log()
    bad = log.copy()
    c = nb1 + nb2 - 32
    if what == "k":
        payload = struct.pack("<QII", 101, 3, 3)
        bad[c + 16: c + 32] = np.frombuffer(payload, dtype=np.uint8)
        bad[c + 12: c + 16] = np.frombuffer(struct.pack("<I", oracle.crc32c(payload)), dtype=np.uint8)
    elif what == "region":
        payload = struct.pack("<QII", 101, 4, 2)
        bad[c + 16: c + 32] = np.frombuffer(payload, dtype=np.uint8)
        bad[c + 12: c + 16] = np.frombuffer(struct.pack("<I", oracle.crc32c(payload)), dtype=np.uint8)
    elif what == "crc":
        bad[c + 20] ^= 1
    elif what == "pageidx":
        bad[c + 4] = 0
    else:
        bad[c + 8] = 32     # a commit header whose len is not 16 (needs 32 bytes to be there: torn instead)
    reg = old.copy()
    st, applied, consumed = oracle.apply_log(bad, nb1 + nb2, [oracle.Region(3, P, reg)])
    if what == "len":
        assert (st, applied, consumed) == (0, 3, nb1)        # len 32 > 16 remaining -> torn
    else:
        assert (st, applied, consumed) == (oracle.ORC_ERR_CORRUPT, 3, nb1)
    assert (reg == mid).all()


def test_duplicates_last_wins_and_multi_region():
    """Config-5a-shaped log written by the oracle's record writer; expected state built by hand."""
    arena = synth.raw_region(1 << 20, 51, "cpu").numpy()
    unit = arena.size // 8
    eps = synth.recovery_epochs(arena.size, 9, 7, 52, forced_repeats=4)
    log = np.zeros(1 << 22, dtype=np.uint8)
    W = 0
    expect = arena.copy()
    views = {}
    for rid, o8, s8, P in synth.C5A_REGIONS:
        views[rid] = (o8 * unit, s8 * unit, P)
    n_rec = 0
    for e in eps:
        o, sz, P = views[e.region_id]
        st, W = oracle.write_epoch(log, W, e.region_id, e.epoch, sz, P, e.pages.numpy(), e.payloads.numpy())
        assert st == 0
        for i, p in enumerate(e.pages.tolist()):
            expect[o + p * P: o + (p + 1) * P] = e.payloads.numpy()[i * P:(i + 1) * P]   # log order, last wins
        n_rec += e.pages.numel()
    reg = arena.copy()
    regions = [oracle.Region(rid, P, reg[o:o + sz]) for rid, (o, sz, P) in views.items()]
    assert oracle.apply_log(log, W, regions) == (0, n_rec, W)
    assert (reg == expect).all()
    # pages did repeat across epochs
    seen, rep = set(), 0
    for e in eps:
        for p in e.pages.tolist():
            rep += (e.region_id, p) in seen
            seen.add((e.region_id, p))
    assert rep >= 4


def test_mixed_regions_in_one_epoch_is_corrupt():
    P = 64
    a = np.zeros(P * 4, dtype=np.uint8)
    b = np.zeros(P * 4, dtype=np.uint8)
    log = np.zeros(1024, dtype=np.uint8)
    pay = np.full(P, 7, dtype=np.uint8)
    # hand-build: record of region 1, record of region 2, commit{region 1, k=2}
    off = 0
    for rid in (1, 2):
        log[off:off + 16] = np.frombuffer(struct.pack("<IIII", rid, 0, P, oracle.crc32c(pay)), dtype=np.uint8)
        log[off + 16: off + 16 + P] = pay
        off += 16 + P
    cp = struct.pack("<QII", 1, 1, 2)
    log[off:off + 16] = np.frombuffer(struct.pack("<IIII", 0xFFFFFFFF, 0xFFFFFFFF, 16, oracle.crc32c(cp)), dtype=np.uint8)
    log[off + 16: off + 32] = np.frombuffer(cp, dtype=np.uint8)
    off += 32
    st, applied, consumed = oracle.apply_log(log, off, [oracle.Region(1, P, a), oracle.Region(2, P, b)])
    assert (st, applied, consumed) == (oracle.ORC_ERR_CORRUPT, 0, 0) and not a.any() and not b.any()


def test_uncommitted_suffix_is_ignored():
    """PAPER.md:L221 "Recovery ignores any suffix without a commit marker"."""
    old, mid, cur, log, nb1, nb2, P = _two_epoch_log()
    reg = old.copy()
    assert oracle.apply_log(log, nb1 + nb2 - 32, [oracle.Region(3, P, reg)]) == (0, 3, nb1)
    assert (reg == mid).all()
