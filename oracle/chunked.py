"""Chunk-wise use of the oracle for regions that do not fit the host twice (TEST INFRASTRUCTURE ONLY).

SURVEY.md 8d: "run parity chunk-wise (stream cur/shadow chunks D2H, oracle per chunk, compare against the matching
slice of the GPU log)".  Nothing here computes anything of the method: every expected byte comes from
``oracle.checkpoint`` (concordia_oracle.c) run on a page-aligned chunk of the region; the only post-processing is
turning the chunk-relative ``page_idx`` header field into the absolute page number (+ first page of the chunk).
The chunks are independent, so the oracle calls run on a thread pool (ctypes releases the GIL); the comparison
against the log is sequential because a chunk's records start where the previous chunk's end.
"""
import struct
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from . import oracle as _o

HDR = 16
COMMIT = 32


def expected_chunk_records(cur_chunk: np.ndarray, shadow_chunk: np.ndarray, P: int, region_id: int, epoch: int, page0: int):
    """oracle.checkpoint on one page-aligned chunk.  Returns (absolute dirty pages as uint32, the chunk's page-record
    bytes with absolute page_idx fields -- no commit record).  shadow_chunk is modified (it becomes cur_chunk)."""
    n = cur_chunk.size
    n_pages = (n + P - 1) // P
    log = np.zeros(n_pages * (HDR + P) + COMMIT, dtype=np.uint8)
    st, D, nb, W = _o.checkpoint(cur_chunk, shadow_chunk, P, region_id, epoch, log, 0)
    assert st == 0
    k = D.size
    if k == 0:
        return D, log[:0]
    body = log[:nb - COMMIT]
    last_len = min(P, n - int(D[-1]) * P)
    n_full = k if last_len == P else k - 1
    if n_full:
        recs = body[:n_full * (HDR + P)].reshape(n_full, HDR + P)
        idx = recs[:, 4:8].copy().view(np.uint32).reshape(n_full)
        assert np.array_equal(idx, D[:n_full])
        recs[:, 4:8] = (idx + np.uint32(page0)).view(np.uint8).reshape(n_full, 4)
    if n_full != k:
        o = n_full * (HDR + P)
        (pi,) = struct.unpack_from("<I", body, o + 4)
        assert pi == int(D[-1])
        struct.pack_into("<I", body, o + 4, pi + page0)
    return D + np.uint32(page0), body


def verify_checkpoint_chunked(N: int, P: int, region_id: int, epoch: int, fetch_cur, fetch_shadow0, fetch_log,
                              chunk_bytes: int = 512 << 20, threads: int = 16, W0: int = 0):
    """Compare a whole checkpoint of a region of N bytes against the oracle, chunk by chunk.

    fetch_cur(o, n) / fetch_shadow0(o, n) -> writable uint8 numpy arrays holding region bytes [o, o+n) after the
    mutation / of the shadow before the checkpoint; fetch_log(o, n) -> uint8 numpy array of log bytes
    [W0 + o, W0 + o + n).  Returns (k, bytes_appended, dirty pages as one uint32 array).  Raises AssertionError with the
    first differing chunk."""
    assert chunk_bytes % P == 0
    offs = list(range(0, N, chunk_bytes))

    def one(o):
        n = min(chunk_bytes, N - o)
        return expected_chunk_records(fetch_cur(o, n), fetch_shadow0(o, n), P, region_id, epoch, o // P)

    pos = 0
    Ds = []
    with ThreadPoolExecutor(max_workers=threads) as ex:
        # a bounded window of chunks in flight keeps host memory at ~3 x threads x chunk_bytes
        for base in range(0, len(offs), threads):
            for o, (D, body) in zip(offs[base:base + threads], ex.map(one, offs[base:base + threads])):
                got = fetch_log(pos, body.size)
                if not np.array_equal(got, body):
                    bad = int(np.nonzero(got != body)[0][0])
                    raise AssertionError("log differs from the oracle in the chunk at region offset %d: log byte %d" % (o, pos + bad))
                pos += body.size
                Ds.append(D)
    D = np.concatenate(Ds) if Ds else np.zeros(0, np.uint32)
    k = int(D.size)
    if k == 0:
        return 0, 0, D
    payload = struct.pack("<QII", epoch, region_id, k)
    commit = struct.pack("<IIII", 0xFFFFFFFF, 0xFFFFFFFF, 16, _o.crc32c(np.frombuffer(payload, np.uint8))) + payload
    got = fetch_log(pos, COMMIT)
    assert got.tobytes() == commit, "commit record differs from the oracle's format"
    return k, pos + COMMIT, D
