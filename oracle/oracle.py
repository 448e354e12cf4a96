"""ctypes front end of oracle/concordia_oracle.c (TEST INFRASTRUCTURE ONLY).

Every function here only marshals numpy buffers into the plain-C oracle; none of
the method's arithmetic lives in Python.  Citations are in concordia_oracle.c.
"""
import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

ORC_OK = 0
ORC_ERR_INVALID = -1
ORC_ERR_LOG_FULL = -4
ORC_ERR_CORRUPT = -5

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "concordia_oracle.c")
_SO = os.path.join(_HERE, "libconcordia_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        subprocess.run(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-pthread", "-o", tmp, _SRC], check=True)
        os.replace(tmp, _SO)
    return _SO


class _CRegion(ctypes.Structure):
    _fields_ = [("region_id", ctypes.c_uint32), ("page_bytes", ctypes.c_uint32), ("bytes", ctypes.c_uint64),
                ("base", ctypes.c_void_p), ("shadow", ctypes.c_void_p)]


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u8p, u32p, u64p = ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint64)
        lib.orc_crc32c.restype = ctypes.c_uint32
        lib.orc_crc32c.argtypes = [u8p, ctypes.c_uint64]
        lib.orc_crc32c_bitwise.restype = ctypes.c_uint32
        lib.orc_crc32c_bitwise.argtypes = [u8p, ctypes.c_uint64]
        lib.orc_scan.restype = ctypes.c_uint64
        lib.orc_scan.argtypes = [u8p, u8p, ctypes.c_uint64, ctypes.c_uint64, u8p]
        lib.orc_scan_mt.restype = ctypes.c_uint64
        lib.orc_scan_mt.argtypes = [u8p, u8p, ctypes.c_uint64, ctypes.c_uint64, u8p, ctypes.c_uint32]
        lib.orc_checkpoint.restype = ctypes.c_int32
        lib.orc_checkpoint.argtypes = [u8p, u8p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint64,
                                       u8p, ctypes.c_uint64, u64p, u32p, u64p, u64p]
        lib.orc_checkpoint_marked.restype = ctypes.c_int32
        lib.orc_checkpoint_marked.argtypes = [u8p, u8p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint32,
                                              ctypes.c_uint64, u8p, ctypes.c_int, ctypes.c_int,
                                              u8p, ctypes.c_uint64, u64p, u32p, u64p, u64p]
        lib.orc_checkpoint_versions.restype = ctypes.c_int32
        lib.orc_checkpoint_versions.argtypes = [u8p, u8p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint32,
                                                ctypes.c_uint64, u8p, u8p,
                                                u8p, ctypes.c_uint64, u64p, u32p, u64p, u64p]
        lib.orc_snapshot.restype = ctypes.c_int32
        lib.orc_snapshot.argtypes = [u8p, u8p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint64,
                                     u8p, ctypes.c_uint64, u64p, u64p, u64p]
        lib.orc_compact_log.restype = ctypes.c_int32
        lib.orc_compact_log.argtypes = [u8p, ctypes.c_uint64, ctypes.POINTER(_CRegion), ctypes.c_uint32,
                                        u8p, ctypes.c_uint64, u64p, u64p, u64p]
        lib.orc_checkpoint_all.restype = ctypes.c_int32
        lib.orc_checkpoint_all.argtypes = [ctypes.POINTER(_CRegion), ctypes.c_uint32, ctypes.c_uint64, u8p, ctypes.c_uint64,
                                           u64p, u8p, u8p, u64p, u64p]
        lib.orc_checkpoint_rle.restype = ctypes.c_int32
        lib.orc_checkpoint_rle.argtypes = [u8p, u8p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint64,
                                           ctypes.c_uint64, u8p, ctypes.c_uint64, u64p, u32p, u64p, u64p, u64p]
        lib.orc_apply.restype = ctypes.c_int32
        lib.orc_apply.argtypes = [u8p, ctypes.c_uint64, ctypes.POINTER(_CRegion), ctypes.c_uint32, u64p, u64p]
        lib.orc_write_epoch.restype = ctypes.c_int32
        lib.orc_write_epoch.argtypes = [u8p, ctypes.c_uint64, u64p, ctypes.c_uint32, ctypes.c_uint64,
                                        ctypes.c_uint64, ctypes.c_uint64, u32p, ctypes.c_uint64, u8p]
        _lib = lib
    return _lib


def _u8(a) -> np.ndarray:
    """View any C-contiguous numpy array (or bytes-like) as a flat uint8 array, no copy."""
    if isinstance(a, (bytes, bytearray, memoryview)):
        a = np.frombuffer(a, dtype=np.uint8)
    a = np.asarray(a)
    if not a.flags["C_CONTIGUOUS"]:
        raise ValueError("oracle buffers must be C-contiguous")
    return a.reshape(-1).view(np.uint8)


def _ptr(a: np.ndarray) -> int:
    return a.ctypes.data


def crc32c(data) -> int:
    d = _u8(data)
    return int(_load().orc_crc32c(_ptr(d), d.size))


def crc32c_bitwise(data) -> int:
    d = _u8(data)
    return int(_load().orc_crc32c_bitwise(_ptr(d), d.size))


def scan(cur, shadow, page_bytes: int) -> np.ndarray:
    """dirty[p] flags (uint8) -- PAPER.md:L261."""
    c, s = _u8(cur), _u8(shadow)
    assert c.size == s.size and page_bytes > 0
    n_pages = (c.size + page_bytes - 1) // page_bytes
    dirty = np.zeros(n_pages, dtype=np.uint8)
    _load().orc_scan(_ptr(c), _ptr(s), c.size, page_bytes, _ptr(dirty))
    return dirty


def scan_mt(cur, shadow, page_bytes: int, n_threads: int) -> np.ndarray:
    c, s = _u8(cur), _u8(shadow)
    assert c.size == s.size and page_bytes > 0
    n_pages = (c.size + page_bytes - 1) // page_bytes
    dirty = np.zeros(n_pages, dtype=np.uint8)
    _load().orc_scan_mt(_ptr(c), _ptr(s), c.size, page_bytes, _ptr(dirty), n_threads)
    return dirty


def checkpoint(cur, shadow, page_bytes: int, region_id: int, epoch: int, log, W: int):
    """One delta checkpoint.  shadow and log are modified in place.

    Returns (status, D, bytes_appended, W_after); D is the ascending uint32 dirty list
    (also returned on LOG_FULL, where nothing was written).
    """
    c, s, lg = _u8(cur), _u8(shadow), _u8(log)
    assert c.size == s.size
    assert s.flags["WRITEABLE"] and lg.flags["WRITEABLE"]
    n_pages = (c.size + page_bytes - 1) // page_bytes
    D = np.zeros(max(n_pages, 1), dtype=np.uint32)
    w = ctypes.c_uint64(W)
    k = ctypes.c_uint64(0)
    nb = ctypes.c_uint64(0)
    st = _load().orc_checkpoint(_ptr(c), _ptr(s), c.size, page_bytes, region_id, epoch,
                                _ptr(lg), lg.size, ctypes.byref(w), _ptr(D), ctypes.byref(k), ctypes.byref(nb))
    return int(st), D[: k.value].copy(), int(nb.value), int(w.value)


def checkpoint_rle(cur, shadow, page_bytes: int, region_id: int, epoch: int, run_pages: int, log, W: int):
    """Delta checkpoint with run records (one record per run of consecutive dirty pages; runs never cross a
    multiple of run_pages).  Returns (status, D, n_runs, bytes_appended, W_after)."""
    c, s, lg = _u8(cur), _u8(shadow), _u8(log)
    assert c.size == s.size
    n_pages = (c.size + page_bytes - 1) // page_bytes
    D = np.zeros(max(n_pages, 1), dtype=np.uint32)
    w, k, runs, nb = ctypes.c_uint64(W), ctypes.c_uint64(0), ctypes.c_uint64(0), ctypes.c_uint64(0)
    st = _load().orc_checkpoint_rle(_ptr(c), _ptr(s), c.size, page_bytes, region_id, epoch, run_pages, _ptr(lg), lg.size,
                                    ctypes.byref(w), _ptr(D), ctypes.byref(k), ctypes.byref(runs), ctypes.byref(nb))
    return int(st), D[: k.value].copy(), int(runs.value), int(nb.value), int(w.value)


def checkpoint_marked(cur, shadow, page_bytes: int, region_id: int, epoch: int, marked, log, W: int,
                      verify: bool = False, consume: bool = False):
    """Allocator-aware checkpoint from a packed dirty-page bitmap (uint32 words, numpy, modified in place
    when consume=True).  shadow may be None when verify=False.  Returns (status, D, bytes_appended, W_after)."""
    c, lg = _u8(cur), _u8(log)
    s = None if shadow is None else _u8(shadow)
    n_pages = (c.size + page_bytes - 1) // page_bytes
    m = np.asarray(marked)
    assert m.dtype == np.uint32 and m.flags["C_CONTIGUOUS"] and m.size >= (n_pages + 31) // 32
    D = np.zeros(max(n_pages, 1), dtype=np.uint32)
    w, k, nb = ctypes.c_uint64(W), ctypes.c_uint64(0), ctypes.c_uint64(0)
    st = _load().orc_checkpoint_marked(_ptr(c), None if s is None else _ptr(s), c.size, page_bytes, region_id, epoch,
                                       _ptr(m), int(verify), int(consume), _ptr(lg), lg.size, ctypes.byref(w),
                                       _ptr(D), ctypes.byref(k), ctypes.byref(nb))
    return int(st), D[: k.value].copy(), int(nb.value), int(w.value)


def checkpoint_versions(cur, shadow, page_bytes: int, region_id: int, epoch: int, version, committed, log, W: int):
    """Allocator-aware checkpoint from per-page version counters (uint64 numpy arrays; ``committed`` is
    advanced in place).  shadow may be None.  Returns (status, D, bytes_appended, W_after)."""
    c, lg = _u8(cur), _u8(log)
    s = None if shadow is None else _u8(shadow)
    n_pages = (c.size + page_bytes - 1) // page_bytes
    v, cm = np.asarray(version), np.asarray(committed)
    assert v.dtype == np.uint64 and cm.dtype == np.uint64 and v.size == n_pages == cm.size
    assert v.flags["C_CONTIGUOUS"] and cm.flags["C_CONTIGUOUS"] and cm.flags["WRITEABLE"]
    D = np.zeros(max(n_pages, 1), dtype=np.uint32)
    w, k, nb = ctypes.c_uint64(W), ctypes.c_uint64(0), ctypes.c_uint64(0)
    st = _load().orc_checkpoint_versions(_ptr(c), None if s is None else _ptr(s), c.size, page_bytes, region_id, epoch,
                                         _ptr(v), _ptr(cm), _ptr(lg), lg.size, ctypes.byref(w),
                                         _ptr(D), ctypes.byref(k), ctypes.byref(nb))
    return int(st), D[: k.value].copy(), int(nb.value), int(w.value)


@dataclass
class Region:
    region_id: int
    page_bytes: int
    base: np.ndarray            # uint8 view, modified in place by apply_log
    shadow: np.ndarray = None   # optional


def apply_log(log, nbytes: int, regions):
    """Replay log[:nbytes] into the regions.  Returns (status, applied, consumed)."""
    lg = _u8(log)
    assert nbytes <= lg.size
    arr = (_CRegion * max(len(regions), 1))()
    keep = []
    for i, r in enumerate(regions):
        b = _u8(r.base)
        assert b.flags["WRITEABLE"]
        keep.append(b)
        sh = 0
        if r.shadow is not None:
            s = _u8(r.shadow)
            assert s.size == b.size and s.flags["WRITEABLE"]
            keep.append(s)
            sh = _ptr(s)
        arr[i] = _CRegion(r.region_id, r.page_bytes, b.size, _ptr(b), sh)
    applied = ctypes.c_uint64(0)
    consumed = ctypes.c_uint64(0)
    st = _load().orc_apply(_ptr(lg), nbytes, arr, len(regions), ctypes.byref(applied), ctypes.byref(consumed))
    return int(st), int(applied.value), int(consumed.value)


def snapshot(cur, shadow, page_bytes: int, region_id: int, epoch: int, log, W: int):
    """Base snapshot: every page of the region as one committed epoch.  shadow (may be None) := cur.
    Returns (status, k, bytes_appended, W_after)."""
    c, lg = _u8(cur), _u8(log)
    s = None if shadow is None else _u8(shadow)
    w, k, nb = ctypes.c_uint64(W), ctypes.c_uint64(0), ctypes.c_uint64(0)
    st = _load().orc_snapshot(_ptr(c), None if s is None else _ptr(s), c.size, page_bytes, region_id, epoch,
                              _ptr(lg), lg.size, ctypes.byref(w), ctypes.byref(k), ctypes.byref(nb))
    return int(st), int(k.value), int(nb.value), int(w.value)


def compact_log(log, nbytes: int, regions, out):
    """Rewrite the committed prefix of log[:nbytes] into `out`: one epoch per region (ascending region id), the last
    record of every page, ascending pages.  Only region_id / page_bytes / size of `regions` are used.
    Returns (status, bytes_out, consumed, n_records_out)."""
    lg, o = _u8(log), _u8(out)
    assert nbytes <= lg.size and o.flags["WRITEABLE"]
    arr = (_CRegion * max(len(regions), 1))()
    for i, r in enumerate(regions):
        b = _u8(r.base)
        arr[i] = _CRegion(r.region_id, r.page_bytes, b.size, _ptr(b), 0)
    nb, consumed, n_out = ctypes.c_uint64(0), ctypes.c_uint64(0), ctypes.c_uint64(0)
    st = _load().orc_compact_log(_ptr(lg), nbytes, arr, len(regions), _ptr(o), o.size, ctypes.byref(nb),
                                 ctypes.byref(consumed), ctypes.byref(n_out))
    return int(st), int(nb.value), int(consumed.value), int(n_out.value)


def checkpoint_all(regions, epoch: int, log, W: int):
    """One boundary: every region that has a shadow is delta-checkpointed in ascending region_id order (base and
    shadow are numpy arrays; shadows and the log are modified in place).
    Returns (status, k per region in the order given, status per region, k_total, bytes_total, W_after)."""
    lg = _u8(log)
    arr = (_CRegion * max(len(regions), 1))()
    keep = []
    for i, r in enumerate(regions):
        b = _u8(r.base)
        keep.append(b)
        sh = 0
        if r.shadow is not None:
            s_ = _u8(r.shadow)
            assert s_.size == b.size and s_.flags["WRITEABLE"]
            keep.append(s_)
            sh = _ptr(s_)
        arr[i] = _CRegion(r.region_id, r.page_bytes, b.size, _ptr(b), sh)
    ks = np.zeros(max(len(regions), 1), dtype=np.uint64)
    sts = np.zeros(max(len(regions), 1), dtype=np.int32)
    w, kt, bt = ctypes.c_uint64(W), ctypes.c_uint64(0), ctypes.c_uint64(0)
    st = _load().orc_checkpoint_all(arr, len(regions), epoch, _ptr(lg), lg.size, ctypes.byref(w), _ptr(ks), _ptr(sts),
                                    ctypes.byref(kt), ctypes.byref(bt))
    return int(st), ks[: len(regions)].tolist(), sts[: len(regions)].tolist(), int(kt.value), int(bt.value), int(w.value)


def write_epoch(log, W: int, region_id: int, epoch: int, region_bytes: int, page_bytes: int, pages, payloads):
    """Append one committed epoch of caller-given page records.  Returns (status, W_after)."""
    lg = _u8(log)
    pg = np.ascontiguousarray(pages, dtype=np.uint32)
    pl = _u8(payloads)
    w = ctypes.c_uint64(W)
    st = _load().orc_write_epoch(_ptr(lg), lg.size, ctypes.byref(w), region_id, epoch, region_bytes, page_bytes,
                                 _ptr(pg), pg.size, _ptr(pl))
    return int(st), int(w.value)
