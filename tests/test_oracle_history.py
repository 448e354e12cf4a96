"""Oracle invariants over long mixed histories (-m "not gpu"): whatever mix of writers produced the log (plain, run-length,
allocator-aware trusted / verified, version counters, snapshot, all-regions), as long as the history ends with a boundary that
diffs every region against its shadow, replaying the log onto the INITIAL state must give the FINAL state, the compacted log
must replay to the same state and be no longer than the original, and every truncation replays, region by region, to a state
that region had at one of the two boundaries around the cut."""
import numpy as np
import pytest

import oracle

SPECS = [(4, 64, 64 * 40 - 16), (9, 256, 256 * 17), (2, 16, 16 * 100)]


def _bitmap(n_pages, pages):
    bm = np.zeros((n_pages + 31) // 32, dtype=np.uint32)
    for p in pages:
        bm[p >> 5] |= np.uint32(1 << (p & 31))
    return bm


@pytest.mark.parametrize("seed", range(8))
def test_replay_of_any_mixed_history_reaches_the_final_state(seed):
    rng = np.random.default_rng(seed)
    R = {}
    for rid, P, N in SPECS:
        cur = rng.integers(0, 256, N, dtype=np.uint8)
        n_pages = (N + P - 1) // P
        R[rid] = dict(P=P, N=N, n=n_pages, cur=cur, sh=cur.copy(), init=cur.copy(),
                      ver=np.zeros(n_pages, np.uint64), com=np.zeros(n_pages, np.uint64))
    regs = [oracle.Region(rid, R[rid]["P"], R[rid]["cur"], R[rid]["sh"]) for rid, _, _ in SPECS]
    log = np.zeros(1 << 20, np.uint8)
    W = 0
    boundaries = [(0, {rid: R[rid]["sh"].copy() for rid in R})]        # (offset, the logged state = shadows) after each call
    for step in range(40):
        for _ in range(int(rng.integers(1, 4))):
            r = R[SPECS[int(rng.integers(0, 3))][0]]
            a = int(rng.integers(0, r["n"]))
            for p in range(a, min(r["n"], a + int(rng.integers(1, 5)))):
                r["cur"][p * r["P"] + int(rng.integers(0, min(r["P"], r["N"] - p * r["P"])))] ^= 0x2B
                r["ver"][p] += np.uint64(1)
        rid = SPECS[int(rng.integers(0, 3))][0]
        r = R[rid]
        op = int(rng.integers(0, 7))
        if op == 0:
            st, _, _, W = oracle.checkpoint(r["cur"], r["sh"], r["P"], rid, step, log, W)
        elif op == 1:
            st, _, _, _, W = oracle.checkpoint_rle(r["cur"], r["sh"], r["P"], rid, step, int(rng.choice([1, 2, 8])), log, W)
        elif op == 2:
            marks = rng.integers(0, r["n"], 6).tolist()
            st, _, _, W = oracle.checkpoint_marked(r["cur"], r["sh"], r["P"], rid, step, _bitmap(r["n"], marks), log, W,
                                                   verify=bool(rng.integers(0, 2)), consume=bool(rng.integers(0, 2)))
        elif op == 3:
            st, _, _, W = oracle.checkpoint_versions(r["cur"], r["sh"], r["P"], rid, step, r["ver"], r["com"], log, W)
        elif op == 4:
            st, _, _, W = oracle.snapshot(r["cur"], r["sh"], r["P"], rid, step, log, W)
        else:
            st, _, _, _, _, W = oracle.checkpoint_all(regs, step, log, W)
        assert st == 0
        boundaries.append((W, {q: R[q]["sh"].copy() for q in R}))
    st, _, _, _, _, W = oracle.checkpoint_all(regs, 99, log, W)          # the closing boundary logs whatever is still unlogged
    assert st == 0
    boundaries.append((W, {q: R[q]["sh"].copy() for q in R}))
    for q in R:
        assert np.array_equal(R[q]["sh"], R[q]["cur"])

    def replay(buf, nbytes):
        state = {q: R[q]["init"].copy() for q in R}
        res = oracle.apply_log(buf, nbytes, [oracle.Region(q, R[q]["P"], state[q]) for q, _, _ in SPECS])
        return res, state

    res, state = replay(log, W)
    assert res[0] == 0 and res[2] == W
    for q in R:
        assert np.array_equal(state[q], R[q]["cur"]), "replay of the full log misses the final state of region %d" % q
    # the compacted log: not longer, same final state, at most one record per page
    out = np.zeros(1 << 20, np.uint8)
    st, nb, consumed, n_out = oracle.compact_log(log, W, [oracle.Region(q, R[q]["P"], R[q]["init"]) for q, _, _ in SPECS], out)
    assert st == 0 and consumed == W and nb <= W and n_out <= sum(R[q]["n"] for q in R)
    res2, state2 = replay(out, nb)
    assert res2 == (0, n_out, nb)
    for q in R:
        assert np.array_equal(state2[q], R[q]["cur"])
    # any truncation replays to the logged state of the last boundary it contains
    offs = [b[0] for b in boundaries]
    for t in sorted(set(rng.integers(0, W + 1, 25).tolist()) | {0, W}):
        res3, state3 = replay(log, t)
        i = max(j for j, o in enumerate(offs) if o <= t)
        nxt = min(i + 1, len(offs) - 1)
        # an all-regions boundary writes one committed epoch per region, so a cut inside it may keep some of them
        assert res3[0] == 0 and offs[i] <= res3[2] <= t and res3[2] <= offs[nxt]
        for q in R:
            assert np.array_equal(state3[q], boundaries[i][1][q]) or np.array_equal(state3[q], boundaries[nxt][1][q]), (t, q)
        if res3[2] == offs[i]:
            for q in R:
                assert np.array_equal(state3[q], boundaries[i][1][q]), (t, q)
