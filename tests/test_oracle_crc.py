"""Pins for the oracle's CRC32C (-m "not gpu").

The oracle's table loop is checked against: the published check value and iSCSI vectors
(tests/golden/crc32c_vectors.txt), its own bit-at-a-time definition, the x86 SSE4.2 crc32
instruction (a hardware implementation of the same polynomial), and CRC theory (linearity,
single-bit sensitivity).
"""
import ctypes
import os
import subprocess

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


def _vectors():
    out = []
    for line in open(os.path.join(HERE, "golden", "crc32c_vectors.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        name, gen, length, exp = [x.strip() for x in line.split("|")]
        n = int(length)
        kind, arg = gen.split(":")
        if kind == "ascii":
            data = np.frombuffer(arg.encode(), dtype=np.uint8)
        elif kind == "fill":
            data = np.full(n, int(arg, 16), dtype=np.uint8)
        elif kind == "inc":
            data = ((int(arg, 16) + np.arange(n)) % 256).astype(np.uint8)
        elif kind == "dec":
            data = ((int(arg, 16) - np.arange(n)) % 256).astype(np.uint8)
        assert data.size == n
        out.append((name, data, int(exp, 16)))
    return out


@pytest.mark.parametrize("name,data,expected", _vectors(), ids=[v[0] for v in _vectors()])
def test_published_vectors(name, data, expected):
    assert oracle.crc32c(data) == expected
    assert oracle.crc32c_bitwise(data) == expected


def test_table_equals_bitwise_random():
    rng = np.random.default_rng(11)
    for n in [1, 2, 3, 15, 16, 17, 255, 256, 4095, 4096, 4097, 65536]:
        d = rng.integers(0, 256, n, dtype=np.uint8)
        assert oracle.crc32c(d) == oracle.crc32c_bitwise(d)


@pytest.fixture(scope="module")
def hwcrc(tmp_path_factory):
    flags = open("/proc/cpuinfo").read()
    if "sse4_2" not in flags:
        pytest.skip("no SSE4.2 on this host")
    so = str(tmp_path_factory.mktemp("hwcrc") / "libhwcrc.so")
    subprocess.run(["gcc", "-O2", "-msse4.2", "-shared", "-fPIC", "-o", so,
                    os.path.join(HERE, "helpers", "hwcrc.c")], check=True)
    lib = ctypes.CDLL(so)
    lib.hw_crc32c.restype = ctypes.c_uint32
    lib.hw_crc32c.argtypes = [ctypes.c_void_p, ctypes.c_uint64]
    return lambda d: int(lib.hw_crc32c(d.ctypes.data, d.size))


def test_against_sse42_instruction(hwcrc):
    rng = np.random.default_rng(12)
    for n in [0, 1, 7, 16, 31, 4096, 16384, 65536, 100003]:
        d = rng.integers(0, 256, n, dtype=np.uint8)
        assert oracle.crc32c(d) == hwcrc(d)


def test_single_bit_flip_changes_crc():
    rng = np.random.default_rng(13)
    d = rng.integers(0, 256, 4096, dtype=np.uint8)
    base = oracle.crc32c(d)
    for byte in [0, 1, 15, 16, 2047, 4080, 4095]:
        for bit in range(8):
            e = d.copy()
            e[byte] ^= np.uint8(1 << bit)
            assert oracle.crc32c(e) != base


def test_affine_linearity():
    # CRC(a) ^ CRC(b) ^ CRC(c) == CRC(a^b^c) for equal-length messages (init/xorout cancel in odd sums)
    rng = np.random.default_rng(14)
    for n in [16, 100, 4096]:
        a, b, c = (rng.integers(0, 256, n, dtype=np.uint8) for _ in range(3))
        assert oracle.crc32c(a) ^ oracle.crc32c(b) ^ oracle.crc32c(c) == oracle.crc32c(a ^ b ^ c)


def test_residue_property():
    # appending the little-endian CRC to the message gives the fixed CRC32C residue
    rng = np.random.default_rng(15)
    res = set()
    for n in [1, 33, 4096]:
        d = rng.integers(0, 256, n, dtype=np.uint8)
        c = oracle.crc32c(d)
        e = np.concatenate([d, np.frombuffer(int(c).to_bytes(4, "little"), dtype=np.uint8)])
        res.add(oracle.crc32c(e))
    assert res == {0x48674BC7}   # CRC32C residue 0xB798B438 after the final XOR
