"""-m "not gpu": oracle/chunked.py (chunk-wise verification used for the 32 / 64 GiB configs) is pinned to the oracle's
own whole-region checkpoint: on regions small enough to checkpoint in one piece, the chunk-wise expectation must
accept exactly the bytes orc_checkpoint writes -- and nothing else."""
import numpy as np
import pytest

import oracle
from oracle import chunked


def _case(N, P, seed, dirty_frac):
    rng = np.random.default_rng(seed)
    cur = rng.integers(0, 256, N, dtype=np.uint8)
    sh = cur.copy()
    n_pages = (N + P - 1) // P
    for p in np.nonzero(rng.random(n_pages) < dirty_frac)[0]:
        plen = min(P, N - p * P)
        sh[p * P + int(rng.integers(0, plen))] ^= 0x40
    return cur, sh


@pytest.mark.parametrize("N,P,chunk,frac", [
    (64 * 256, 256, 4 * 256, 0.3),            # 16 chunks
    (64 * 256, 256, 4 * 256, 1.0),            # all dirty
    (64 * 256 - 112, 256, 8 * 256, 1.0),      # short last page in the last chunk
    (64 * 256 - 112, 256, 8 * 256, 0.1),
    (10 * 4096, 4096, 3 * 4096, 0.5),         # ragged last chunk
    (5 * 1024, 1024, 8 * 1024, 1.0),          # one chunk
    (16 * 64, 64, 64, 0.0),                   # nothing dirty
])
def test_chunked_expectation_equals_whole_region_oracle(N, P, chunk, frac):
    cur, sh0 = _case(N, P, N + P, frac)
    n_pages = (N + P - 1) // P
    whole = np.zeros(n_pages * (16 + P) + 32 + 64, np.uint8)
    sh = sh0.copy()
    st, D, nb, W = oracle.checkpoint(cur, sh, P, 9, 1234567890123, whole, 0)
    assert st == 0
    k, nbytes, Dc = chunked.verify_checkpoint_chunked(
        N, P, 9, 1234567890123, lambda o, n: cur[o:o + n].copy(), lambda o, n: sh0[o:o + n].copy(),
        lambda o, n: whole[o:o + n], chunk_bytes=chunk, threads=3)
    assert (k, nbytes) == (D.size, nb) and Dc.tolist() == D.tolist()
    if k:
        # any single corrupted byte of the log is caught (payload, header field, commit record)
        rng = np.random.default_rng(1)
        for pos in [0, 4, 8, 12, 16, nb - 1, nb - 20, nb - 32] + rng.integers(0, nb, 6).tolist():
            bad = whole.copy()
            bad[pos] ^= 0x01
            with pytest.raises(AssertionError):
                chunked.verify_checkpoint_chunked(N, P, 9, 1234567890123, lambda o, n: cur[o:o + n].copy(),
                                                  lambda o, n: sh0[o:o + n].copy(), lambda o, n: bad[o:o + n],
                                                  chunk_bytes=chunk, threads=2)
