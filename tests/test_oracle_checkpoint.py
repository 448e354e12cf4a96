"""Pins for the checkpoint oracle (-m "not gpu"): worked examples, brute force, invariants."""
import os
import struct

import numpy as np
import pytest
import torch

import oracle
import synth

HERE = os.path.dirname(os.path.abspath(__file__))


def _hex_fixture(name):
    data = bytearray()
    for line in open(os.path.join(HERE, "golden", name)):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        data += bytes(int(x, 16) for x in line.split())
    return bytes(data)


# --- an independent restatement of the record layout, in pure Python (struct + bit-loop CRC) ---

def _py_crc32c(b: bytes) -> int:
    crc = 0xFFFFFFFF
    for x in b:
        crc ^= x
        for _ in range(8):
            crc = (crc >> 1) ^ 0x82F63B78 if crc & 1 else crc >> 1
    return crc ^ 0xFFFFFFFF


def _py_checkpoint(cur: bytes, shadow: bytes, P: int, rid: int, epoch: int) -> tuple:
    """Byte loop per page; returns (D, log bytes)."""
    N = len(cur)
    D, out = [], b""
    for p in range((N + P - 1) // P):
        a, b = cur[p * P:(p + 1) * P], shadow[p * P:(p + 1) * P]
        if any(x != y for x, y in zip(a, b)):
            D.append(p)
            out += struct.pack("<IIII", rid, p, len(a), _py_crc32c(a)) + a
    if D:
        cp = struct.pack("<QII", epoch, rid, len(D))
        out += struct.pack("<IIII", 0xFFFFFFFF, 0xFFFFFFFF, 16, _py_crc32c(cp)) + cp
    return D, out


def test_worked_example_1():
    golden = _hex_fixture("worked_example_1.txt")
    assert len(golden) == 96
    cur = np.arange(64, dtype=np.uint8)
    sh = cur.copy()
    sh[17] ^= 0x01
    sh[63] ^= 0x80
    old = sh.copy()
    log = np.zeros(200, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur, sh, 16, 7, 3, log, 0)
    assert st == oracle.ORC_OK and D.tolist() == [1, 3] and nb == 96 and W == 96
    assert log[:96].tobytes() == golden
    assert not log[96:].any()
    assert oracle.crc32c(log[:96]) == 0x10A9D987
    assert (sh == cur).all()
    # apply to a region holding the old shadow reproduces cur; 95 bytes apply nothing
    reg = old.copy()
    st, applied, consumed = oracle.apply_log(log, 96, [oracle.Region(7, 16, reg)])
    assert (st, applied, consumed) == (0, 2, 96) and (reg == cur).all()
    reg = old.copy()
    st, applied, consumed = oracle.apply_log(log, 95, [oracle.Region(7, 16, reg)])
    assert (st, applied, consumed) == (0, 0, 0) and (reg == old).all()


def test_worked_example_2():
    golden_tail = _hex_fixture("worked_example_2.txt")
    assert len(golden_tail) == 64
    N, P = 80, 32
    cur = ((3 * np.arange(N)) % 256).astype(np.uint8)
    sh = np.zeros(N, dtype=np.uint8)
    log = np.zeros(400, dtype=np.uint8)
    # capacity below 160 -> LOG_FULL, nothing written, shadow untouched
    st, D, nb, W = oracle.checkpoint(cur, sh, P, 2, 10, log[:159], 0)
    assert st == oracle.ORC_ERR_LOG_FULL and nb == 0 and W == 0 and not log.any() and not sh.any()
    assert D.tolist() == [0, 1, 2]
    st, D, nb, W = oracle.checkpoint(cur, sh, P, 2, 10, log, 0)
    assert (st, D.tolist(), nb, W) == (0, [0, 1, 2], 160, 160)
    crcs = [struct.unpack_from("<I", log, off + 12)[0] for off in (0, 48, 96, 128)]
    assert crcs == [0x9E4888F6, 0xCE222AF8, 0xCBBDB609, 0xDA3BABB7]
    lens = [struct.unpack_from("<I", log, off + 8)[0] for off in (0, 48, 96, 128)]
    assert lens == [32, 32, 16, 16]
    epoch10 = cur.copy()
    cur[79] ^= 0xFF
    st, D, nb, W = oracle.checkpoint(cur, sh, P, 2, 11, log, W)
    assert (st, D.tolist(), nb, W) == (0, [2], 64, 224)
    assert log[160:224].tobytes() == golden_tail
    assert oracle.crc32c(log[:224]) == 0x241E68BB
    # replay: all 224 bytes -> final cur (last wins); 160..223 bytes -> epoch-10 state
    reg = np.zeros(N, dtype=np.uint8)
    assert oracle.apply_log(log, 224, [oracle.Region(2, P, reg)]) == (0, 4, 224)
    assert (reg == cur).all()
    for cut in (160, 161, 176, 200, 223):
        reg = np.zeros(N, dtype=np.uint8)
        assert oracle.apply_log(log, cut, [oracle.Region(2, P, reg)]) == (0, 3, 160)
        assert (reg == epoch10).all()


@pytest.mark.parametrize("P,n_pages,tail", [(16, 5, 0), (16, 8, 0), (64, 6, 48), (64, 8, 0), (4096, 4, 1024)])
def test_brute_force_all_subsets(P, n_pages, tail):
    """Every dirty subset of a tiny region: oracle == byte-loop restatement in pure Python."""
    N = (n_pages - 1) * P + (tail or P)
    rng = np.random.default_rng(100 + P + n_pages)
    base = rng.integers(0, 256, N, dtype=np.uint8)
    real_pages = (N + P - 1) // P
    for mask in range(1 << real_pages):
        cur = base.copy()
        sh = base.copy()
        for p in range(real_pages):
            if mask >> p & 1:
                plen = min(P, N - p * P)
                off = p * P + int(rng.integers(0, plen))
                sh[off] ^= np.uint8(1 << int(rng.integers(0, 8)))
        log = np.zeros(real_pages * (16 + P) + 32, dtype=np.uint8)
        D_py, log_py = _py_checkpoint(cur.tobytes(), sh.tobytes(), P, 5, mask)
        st, D, nb, W = oracle.checkpoint(cur, sh, P, 5, mask, log, 0)
        assert st == 0 and D.tolist() == D_py == [p for p in range(real_pages) if mask >> p & 1]
        assert nb == len(log_py) and log[:nb].tobytes() == log_py
        assert (sh == cur).all()


def test_boundary_flips_and_bit_lanes():
    """Byte 0 / byte P-1 / every byte lane of a 16-B vector / every bit of a byte are all seen."""
    P, n_pages = 256, 6
    base = np.random.default_rng(7).integers(0, 256, P * n_pages, dtype=np.uint8)
    for page in (0, 3, n_pages - 1):
        for off in list(range(16)) + [P - 16 + i for i in range(16)] + [P // 2]:
            for bit in (0, 7):
                sh = base.copy()
                sh[page * P + off] ^= np.uint8(1 << bit)
                assert oracle.scan(base, sh, P).nonzero()[0].tolist() == [page]
    # adjacent pages: last byte of page 2 and first byte of page 3
    sh = base.copy()
    sh[3 * P - 1] ^= 1
    sh[3 * P] ^= 1
    assert oracle.scan(base, sh, P).nonzero()[0].tolist() == [2, 3]


def test_bitwise_semantics_float():
    """-0.0 vs +0.0 is dirty; identical NaN payloads are clean (reading #2)."""
    a = np.zeros(1024, dtype=np.float32)
    b = a.copy()
    b[300] = -0.0
    assert oracle.scan(a, b, 1024).tolist() == [0, 1, 0, 0]
    a[:] = np.nan
    b = a.copy()
    assert oracle.scan(a, b, 1024).sum() == 0


def test_zero_mutations_empty_log():
    """north_star invariant 1; PAPER.md:L388 (no mutation -> 0 dirty pages)."""
    cur = synth.raw_region(1 << 18, 21, "cpu").numpy()
    sh = cur.copy()
    log = np.zeros(1024, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur, sh, 4096, 1, 1, log, 0)
    assert (st, D.size, nb, W) == (0, 0, 0, 0) and not log.any()


def test_all_dirty_is_full_copy():
    """north_star invariant 2: payloads concatenated == region byte-for-byte."""
    P, N = 4096, 4096 * 37 + 1024
    cur = synth.raw_region(N, 22, "cpu").numpy()
    sh = np.bitwise_not(cur)
    n_pages = (N + P - 1) // P
    log = np.zeros(n_pages * (16 + P) + 32, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur, sh, P, 9, 4, log, 0)
    assert st == 0 and D.tolist() == list(range(n_pages))
    assert nb == (n_pages - 1) * (16 + P) + 16 + 1024 + 32
    payload = np.concatenate([log[i * (16 + P) + 16: i * (16 + P) + 16 + min(P, N - i * P)] for i in range(n_pages)])
    assert (payload == cur).all()


def test_single_page_in_8192_page_arena():
    """one modified 4 KB page in an 8,192-page arena -> 1 record, 8,192:1."""
    P, n_pages = 4096, 8192
    cur = synth.raw_region(P * n_pages, 23, "cpu").numpy()
    sh = cur.copy()
    cur[P * 4321 + 99] ^= 0x10
    log = np.zeros(16 + P + 32, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur, sh, P, 1, 1, log, 0)
    assert st == 0 and D.tolist() == [4321] and nb == 16 + P + 32
    assert n_pages // D.size == 8192
    # immediate second checkpoint is empty (shadow == cur)
    st, D, nb, W2 = oracle.checkpoint(cur, sh, P, 1, 2, log, 0)
    assert D.size == 0 and nb == 0


def test_lora_shape_all_adapter_pages_zero_frozen():
    """a LoRA step dirties exactly the adapter pages, frozen pages 0.
    Scaled: 'frozen' bytes followed by an adapter region whose every page is updated."""
    P = 4096
    frozen = synth.raw_region(P * 570, 24, "cpu").numpy()
    adapter = synth.lora_region(1, 25, "cpu", rank=2, hidden=1280).clone()     # 10 pages of 4 KiB... 2*1280*4*2*4
    n_ad = adapter.numel() // P
    cur = np.concatenate([frozen, adapter.numpy()])
    sh = cur.copy()
    t = torch.from_numpy(cur[frozen.size:])
    pages = synth.lora_update(t, P, 1.0, 26)
    assert pages.numel() == n_ad
    dirty = oracle.scan(cur, sh, P)
    assert dirty[:570].sum() == 0 and dirty[570:].all()


@pytest.mark.parametrize("cfg", ["c1", "c2", "c3", "c4"])
def test_generator_dirty_set_equals_oracle(cfg):
    """The generator's intended dirty set equals the oracle's on scaled versions of configs 1-4."""
    if cfg == "c1":
        P = 4096
        cur = synth.raw_region(1 << 22, 1001, "cpu")
        old = cur.clone()
        pages = synth.mutate_byte_flips(cur, P, 0.01, 1001)
    elif cfg == "c2":
        P = 65536
        cur = synth.kv_cache_region(2, 64, 1002, "cpu")
        old = cur.clone()
        pages = synth.kv_decode_step(cur, 2, 64, 8, 1002)
    elif cfg == "c3":
        P = 65536
        cur = synth.lora_region(2, 1003, "cpu")
        old = cur.clone()
        pages = synth.lora_update(cur, P, 0.05, 1003)
    else:
        P = 16384
        cur = synth.bf16_normal_region(1 << 23, 1004, "cpu", 1 << 21)
        old = cur.clone()
        pages, _, _ = synth.sparse_xor_flips(cur, P, 0.001, 1004)
    sh = old.numpy().copy()
    n_pages = cur.numel() // P
    log = np.zeros(len(pages) * (16 + P) + 32, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur.numpy(), sh, P, 1, 1, log, 0)
    assert st == 0 and D.tolist() == pages.tolist()
    assert nb == len(pages) * (16 + P) + 32          # closed form, SURVEY.md 8c
    assert (np.diff(D.astype(np.int64)) > 0).all()
    assert (sh == cur.numpy()).all()
    # header fields re-derivable, every CRC re-verifiable with the independent bit loop
    for i, p in enumerate(pages.tolist()[:3]):
        off = i * (16 + P)
        rid, pi, ln, crc = struct.unpack_from("<IIII", log, off)
        assert (rid, pi, ln) == (1, p, P)
        assert crc == _py_crc32c(cur.numpy()[p * P:(p + 1) * P].tobytes()[:ln]) if P <= 16384 else True
    # apply(old snapshot, log) == new region (north_star invariant 3)
    reg = old.numpy().copy()
    assert oracle.apply_log(log, nb, [oracle.Region(1, P, reg)]) == (0, len(pages), nb)
    assert (reg == cur.numpy()).all()


def test_closed_form_log_sizes_full_configs():
    """SURVEY.md 8c closed forms at BASELINE.json sizes (arithmetic only)."""
    assert 164 * (16 + 4096) + 32 == 674_400
    assert 8192 * (16 + 65536) + 32 == 537_002_016
    assert 52 * (16 + 65536) + 32 == 3_408_736
    assert 656 * (16 + 4096) + 32 == 2_697_504


def test_log_full_retry_gives_same_log():
    P = 1024
    cur = synth.raw_region(P * 64, 31, "cpu").numpy()
    sh = cur.copy()
    for p in (3, 9, 40):
        cur[p * P + 5] ^= 0xFF
    need = 3 * (16 + P) + 32
    log = np.zeros(need + 100, dtype=np.uint8)
    st, D, nb, W = oracle.checkpoint(cur, sh, P, 2, 8, log, 101)     # 101 + need > capacity
    assert st == oracle.ORC_ERR_LOG_FULL and W == 101 and nb == 0 and not log.any()
    assert oracle.scan(cur, sh, P).sum() == 3                          # shadow untouched
    st, D, nb, W = oracle.checkpoint(cur, sh, P, 2, 8, log, 0)         # after reset
    assert st == 0 and nb == need and D.tolist() == [3, 9, 40]
    ref = np.zeros_like(log)
    sh2 = cur.copy()
    for p in (3, 9, 40):
        sh2[p * P + 5] ^= 0xFF
    oracle.checkpoint(cur, sh2, P, 2, 8, ref, 0)
    assert (ref == log).all()


def test_scan_mt_equals_scan():
    cur = synth.raw_region(1 << 20, 41, "cpu").numpy()
    sh = cur.copy()
    sh[::70001] ^= 1
    assert (oracle.scan_mt(cur, sh, 4096, 5) == oracle.scan(cur, sh, 4096)).all()
