"""GPU: ring buffer + persistent worker.  Same log bytes as the host-launched path and the oracle;
FIFO completion; ring-full; wrap-around; liveness."""
import time

import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2606_23521_b200 as cc

pytestmark = pytest.mark.gpu


def _mk(P=4096, n_pages=512, cap=8, seed=1006, log_bytes=1 << 22, pinned=True, **kw):
    cur = synth.raw_region(P * n_pages, seed, "cuda")
    ctx = cc.Context(ring_capacity=cap, max_lifetime_ns=int(60e9), **kw)
    sh = ctx.register_region(1, cur, P)
    log = torch.zeros(log_bytes, dtype=torch.uint8, pin_memory=True) if pinned else \
        torch.zeros(log_bytes, dtype=torch.uint8, device="cuda")
    committed = torch.zeros(1, dtype=torch.int64, pin_memory=True)
    ctx.log_attach(log, committed)
    ctx.apply_attach(4096)
    return ctx, cur, sh, log, committed


def test_nop_roundtrip_alive_and_stop():
    ctx, cur, sh, log, committed = _mk()
    assert not ctx.worker_alive()
    with pytest.raises(cc.ConcordiaError) as e:
        ctx.submit(cc.CC_TASK_NOP)
    assert e.value.code == cc.CC_ERR_WORKER
    ctx.worker_start()
    try:
        assert ctx.worker_alive()
        seqs = [ctx.submit(cc.CC_TASK_NOP) for _ in range(5)]
        assert seqs == list(range(5))
        for s in seqs:
            r = ctx.wait(s, 5.0)
            assert r.seq_done == s + 1 and r.status == 0 and r.flags == cc.CC_TASK_NOP
        h, t = ctx.peek_queue()
        assert (h, t) == (5, 5)
        with pytest.raises(cc.ConcordiaError) as e:          # registration only while stopped
            ctx.log_reset()
        assert e.value.code == cc.CC_ERR_WORKER
    finally:
        ctx.worker_stop()
    assert not ctx.worker_alive()
    ctx.log_reset()
    ctx.shutdown()


def test_wraparound_ring_full_and_fifo():
    ctx, cur, sh, log, committed = _mk(cap=4)
    ctx.worker_start()
    try:
        done = []
        full_seen = 0
        submitted = 0
        while submitted < 40:
            try:
                s = ctx.submit(cc.CC_TASK_NOP)
                submitted += 1
                done.append(s)
            except cc.ConcordiaError as e:
                assert e.code == cc.CC_ERR_RING_FULL
                full_seen += 1
                h, t = ctx.peek_queue()
                ctx.wait(h, 5.0) if h < t else None
        last_end = 0
        r = ctx.wait(done[-1], 5.0)
        assert r.seq_done == 40
        h, t = ctx.peek_queue()
        assert (h, t) == (40, 40)
    finally:
        ctx.worker_stop()
    ctx.shutdown()


@pytest.mark.parametrize("fused", [False, True])
def test_worker_checkpoint_equals_host_launched_and_oracle(fused):
    """C5b-shaped: MUTATE -> DELTA_CKPT tasks; parity of every task's log bytes on the first tasks.
    fused: the tasks carry CC_TASKF_FUSED (single fused pass inside the worker)."""
    fl = cc.CC_TASKF_FUSED if fused else 0
    P, n_pages, n_mut = 4096, 512, 6
    ctx, cur, sh, log, committed = _mk(P=P, n_pages=n_pages, cap=64)
    host_cur = cur.cpu().numpy().copy()
    host_sh = host_cur.copy()
    olog = np.zeros(log.numel(), dtype=np.uint8)
    W = 0
    ctx.worker_start()
    try:
        pend = []
        for task in range(16):
            pages, h = synth.worker_mutation_pages(task, n_pages, n_mut, 1006)
            A = 2 * ((1006 * 7919 + 12345) % 100000) + 1
            ctx.submit(cc.CC_TASK_TEST_MUTATE, region_id=1, arg0=n_mut, arg1=A, arg2=h)
            s = ctx.submit(cc.CC_TASK_DELTA_CKPT, region_id=1, epoch=1000 + task, flags=fl)
            for j, p in enumerate(pages):
                host_cur[p * P + (h + j) % P] ^= 0x5A
            st, D, nb, W = oracle.checkpoint(host_cur, host_sh, P, 1, 1000 + task, olog, W)
            pend.append((s, D.size, nb, W))
        for s, k, nb, w in pend:
            r = ctx.wait(s, 10.0)
            assert (r.status, r.n_dirty, r.bytes, r.log_offset_after, r.epoch) == (0, k, nb, w, 1000 + (s // 2))
            assert r.t_end_ns >= r.t_start_ns
        assert int(committed.item()) == W
        assert np.array_equal(log.numpy(), olog)
        # log reset through the ring, then one more checkpoint lands at offset 0
        ctx.submit(cc.CC_TASK_LOG_RESET)
        ctx.submit(cc.CC_TASK_TEST_MUTATE, region_id=1, arg0=1, arg1=1, arg2=7)
        s = ctx.submit(cc.CC_TASK_DELTA_CKPT, region_id=1, epoch=5, flags=fl)
        r = ctx.wait(s, 10.0)
        assert (r.n_dirty, r.bytes, r.log_offset_after) == (1, 16 + P + 32, 16 + P + 32)
        # unknown region -> NOT_REGISTERED, worker keeps running
        s = ctx.submit(cc.CC_TASK_DELTA_CKPT, region_id=77, epoch=6)
        assert ctx.wait(s, 10.0).status == cc.CC_ERR_NOT_REGISTERED
        assert ctx.worker_alive()
    finally:
        ctx.worker_stop()
    # after the worker has left, the host-launched path continues on the same state
    torch.cuda.synchronize()
    assert np.array_equal(sh.cpu().numpy(), cur.cpu().numpy())
    ctx.shutdown()


def test_worker_restore_task():
    P, n_pages = 4096, 256
    ctx, cur, sh, log, committed = _mk(P=P, n_pages=n_pages, cap=16, pinned=True)
    old = cur.clone()
    for p in (0, 100, 255):
        cur[p * P + 17] ^= 0x33
    new = cur.clone()
    res = cc.Result()
    ctx.checkpoint_delta(1, 1, res)
    torch.cuda.synchronize()
    nb = res.read().bytes
    assert nb == 3 * (16 + P) + 32
    cur.copy_(old)
    sh.copy_(old)
    torch.cuda.synchronize()
    ctx.worker_start()
    try:
        s = ctx.submit(cc.CC_TASK_RESTORE, arg0=log.data_ptr(), arg1=nb)
        r = ctx.wait(s, 10.0)
        assert (r.status, r.n_dirty, r.bytes, r.epoch) == (0, 3, nb, 1)
    finally:
        ctx.worker_stop()
    torch.cuda.synchronize()
    assert torch.equal(cur, new) and torch.equal(sh, new)
    ctx.shutdown()


def test_worker_lifetime_watchdog():
    """The worker leaves by itself after max_lifetime_ns (safety net against a lost host)."""
    cur = synth.raw_region(4096 * 8, 3, "cuda")
    ctx = cc.Context(ring_capacity=4, max_lifetime_ns=int(0.3e9))
    ctx.register_region(1, cur, 4096)
    ctx.worker_start()
    time.sleep(1.0)
    assert not ctx.worker_alive()
    ctx.worker_stop()
    ctx.shutdown()


def test_measurement_hooks():
    """cc_measure_submit_cost / cc_measure_launch_cost return sane numbers and leave the ring consistent."""
    ctx, cur, sh, log, committed = _mk(cap=16)
    with pytest.raises(cc.ConcordiaError):
        ctx.measure_submit_cost(10)                     # needs a running worker
    a, b = ctx.measure_launch_cost(200)
    assert 0 < b < 1e6 and 0 < a < 1e6                  # ns per launch: batched, and with a sync per launch
    ctx.worker_start()
    try:
        ns = ctx.measure_submit_cost(5000)              # many more than the ring holds
        assert 0 < ns < 20000
        h, t = ctx.peek_queue()
        assert h == t == 5000
        s = ctx.submit(cc.CC_TASK_NOP)
        assert ctx.wait(s, 10.0).status == 0 and s == 5000
    finally:
        ctx.worker_stop()
    ctx.shutdown()


def test_recovery_tasks_without_apply_scratch_are_refused():
    """RESTORE / COMPACT_LOG on a worker started without cc_apply_attach used to store through a
    null table pointer; they must answer CC_ERR_INVALID, as must null / misaligned log pointers."""
    cur = synth.raw_region(4096 * 64, 7, "cuda")
    ctx = cc.Context(ring_capacity=8, max_lifetime_ns=int(30e9))
    ctx.register_region(1, cur, 4096)
    log = torch.zeros(1 << 16, dtype=torch.uint8, device="cuda")
    out = torch.zeros(1 << 16, dtype=torch.uint8, device="cuda")
    ctx.log_attach(log)
    ctx.worker_start()                                      # no apply_attach
    try:
        for kind, args in ((cc.CC_TASK_RESTORE, dict(arg0=log.data_ptr(), arg1=64)),
                           (cc.CC_TASK_COMPACT_LOG, dict(arg0=log.data_ptr(), arg1=64, arg2=out.data_ptr(), arg3=out.numel()))):
            r = ctx.wait(ctx.submit(kind, **args), 10.0)
            assert r.status == cc.CC_ERR_INVALID, (kind, r.as_dict())
        assert ctx.worker_alive()                           # the resident kernel survived
        r = ctx.wait(ctx.submit(cc.CC_TASK_NOP), 5.0)
        assert r.status == 0
    finally:
        ctx.worker_stop()
    ctx.apply_attach(256)
    ctx.worker_start()
    try:
        for args in (dict(arg0=0, arg1=64), dict(arg0=log.data_ptr() + 8, arg1=64)):
            r = ctx.wait(ctx.submit(cc.CC_TASK_RESTORE, **args), 10.0)
            assert r.status == cc.CC_ERR_INVALID, r.as_dict()
        r = ctx.wait(ctx.submit(cc.CC_TASK_COMPACT_LOG, arg0=log.data_ptr(), arg1=4096, arg2=log.data_ptr() + 1024, arg3=4096), 10.0)
        assert r.status == cc.CC_ERR_INVALID                # overlapping input / output
        r = ctx.wait(ctx.submit(cc.CC_TASK_RESTORE, arg0=log.data_ptr(), arg1=0), 10.0)
        assert (r.status, r.n_dirty, r.bytes) == (0, 0, 0)  # an empty log is a valid log
    finally:
        ctx.worker_stop()
    ctx.shutdown()


def test_host_launched_calls_are_refused_while_the_worker_runs():
    """the host-launched data path shares control blocks with the resident worker."""
    ctx, cur, sh, log, committed = _mk()
    res = cc.Result()
    marks = torch.zeros(16, dtype=torch.int32, device="cuda")
    ctx.worker_start()
    try:
        calls = [lambda: ctx.checkpoint_delta(1, 1, res), lambda: ctx.checkpoint_delta_fused(1, 1, res),
                 lambda: ctx.checkpoint_delta_rle(1, 1, 4, res), lambda: ctx.checkpoint_marked(1, 1, marks, 0, res),
                 lambda: ctx.checkpoint_all(1, res), lambda: ctx.snapshot_region(1, 1, res), lambda: ctx.scan_only(1, res),
                 lambda: ctx.apply_log(log, 0, res)]
        for c in calls:
            with pytest.raises(cc.ConcordiaError) as e:
                c()
            assert e.value.code == cc.CC_ERR_WORKER
    finally:
        ctx.worker_stop()
    ctx.checkpoint_delta(1, 1, res)
    torch.cuda.synchronize()
    assert res.read().status == 0
    ctx.shutdown()


def test_wait_and_submit_notice_a_worker_that_left_by_itself():
    """after max_lifetime_ns the kernel exits; cc_wait must not spin to its timeout and cc_submit must
    stop accepting tasks."""
    cur = synth.raw_region(4096 * 64, 8, "cuda")
    ctx = cc.Context(ring_capacity=4, max_lifetime_ns=int(0.3e9))
    ctx.register_region(1, cur, 4096)
    ctx.worker_start()
    time.sleep(0.6)                                         # the worker's lifetime is over
    t0 = time.time()
    got = None
    try:
        for _ in range(8):                                  # at most `capacity` submissions go through, then WORKER
            s = ctx.submit(cc.CC_TASK_NOP)
            ctx.wait(s, 20.0)
    except cc.ConcordiaError as e:
        got = e.code
    assert got == cc.CC_ERR_WORKER, got
    assert time.time() - t0 < 5.0                           # not the 20 s timeout
    assert not ctx.worker_alive()
    ctx.shutdown()


def test_two_host_threads_submitting_at_once(tmp_path):
    """SURVEY.md section 5 row 2 / PAPER.md:L119, L249: the ring has ONE producer.  Two native threads call cc_submit
    on the same context as fast as they can (100,000 NOP tasks in all, the ring mostly full): a thread that finds the
    other one inside is refused with CC_ERR_INVALID and tries again; no sequence number is handed out twice or skipped,
    each thread's numbers ascend, every task completes, and the completion records of the last ring's worth of tasks
    carry the tag of the thread that really submitted them."""
    import ctypes
    import os
    import subprocess
    so = str(tmp_path / "libring_stress.so")
    subprocess.run(["gcc", "-O2", "-pthread", "-shared", "-fPIC", "-o", so,
                    os.path.join(os.path.dirname(os.path.abspath(__file__)), "helpers", "ring_stress.c")], check=True)
    h = ctypes.CDLL(so)
    h.ring_stress.restype = ctypes.c_int32
    h.ring_stress.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    n, cap = 50_000, 256
    ctx = cc.Context(ring_capacity=cap)
    ctx.worker_start()
    try:
        sa, sb = np.zeros(n, np.uint64), np.zeros(n, np.uint64)
        cnt = np.zeros(4, np.uint64)
        submit = ctypes.cast(ctx.lib.cc_submit, ctypes.c_void_p)
        rc = h.ring_stress(submit, ctx.h, n, sa.ctypes.data, sb.ctypes.data, cnt.ctypes.data)
        assert rc == 0, rc
        assert np.all(np.diff(sa.astype(np.int64)) > 0) and np.all(np.diff(sb.astype(np.int64)) > 0)
        both = np.sort(np.concatenate([sa, sb]))
        assert np.array_equal(both, np.arange(2 * n, dtype=np.uint64)), "a sequence number was lost or handed out twice"
        last = ctx.wait(2 * n - 1, 30.0)
        assert last.status == 0 and last.seq_done == 2 * n
        assert ctx.peek_queue() == (2 * n, 2 * n)
        owner = {int(s): (1, i) for i, s in enumerate(sa)}
        owner.update({int(s): (2, i) for i, s in enumerate(sb)})
        for seq in range(2 * n - cap, 2 * n):
            r = ctx.poll(seq)
            tag, i = owner[seq]
            assert r is not None and r.seq_done == seq + 1 and r.epoch == (tag << 32) | i, (seq, r.as_dict())
        if (os.cpu_count() or 1) >= 2:
            assert int(cnt[0] + cnt[1]) > 0, "the two producers never met inside cc_submit: %s" % cnt.tolist()
        assert ctx.worker_alive()
    finally:
        ctx.worker_stop()
        ctx.shutdown()
