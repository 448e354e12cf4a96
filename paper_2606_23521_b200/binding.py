"""Thin ctypes binding of libconcordia.so -- argument marshalling only.

Every step of the path (scan, compaction, gather + CRC32C, commit, shadow update, apply, ring
worker) runs in the CUDA kernels behind the C ABI of include/concordia.h.  PyTorch is used for
device memory, pinned memory and streams.  There is no CPU fallback: importing works without a
GPU (so that the symbol table can be checked), but creating a Context without the library or
without a CUDA device raises.
"""
import ctypes

import torch

from . import build as _build

CC_OK = 0
CC_PENDING = 1
CC_ERR_INVALID = -1
CC_ERR_NOT_REGISTERED = -2
CC_ERR_EXISTS = -3
CC_ERR_LOG_FULL = -4
CC_ERR_CORRUPT = -5
CC_ERR_RING_FULL = -6
CC_ERR_WORKER = -7
CC_ERR_CUDA = -8
CC_ERR_TIMEOUT = -9
CC_ERR_SCRATCH = -10
CC_ERR_STATIC_LIMIT = -11
CC_STATIC_MAX_PAGES = 1 << 24

CC_REG_SNAPSHOT_NOW = 1
CC_REG_NO_SHADOW = 2
CC_MARK_VERIFY = 1
CC_MARK_CONSUME = 2

CC_TASK_NOP = 0
CC_TASK_DELTA_CKPT = 1
CC_TASK_RESTORE = 2
CC_TASK_LOG_RESET = 3
CC_TASK_TEST_MUTATE = 4
CC_TASK_MARKED_CKPT = 5
CC_TASK_VERSION_CKPT = 6
CC_TASK_SNAPSHOT = 7
CC_TASK_COMPACT_LOG = 8
CC_TASK_CKPT_ALL = 9
CC_TASK_EXIT = 255
CC_TASKF_FUSED = 1
CC_TASKF_RLE = 2

CC_WORKER_BLOCKS_DEFAULT = 16
CC_WORKER_BLOCKS_ALL = 0xFFFFFFFF
CC_DISC_SCAN, CC_DISC_MARKS, CC_DISC_VERSIONS, CC_DISC_ALL = 0, 1, 3, 4
CC_PATH_AUTO, CC_PATH_SINGLE_PASS, CC_PATH_PHASES, CC_PATH_SMALL = 0, 1, 2, 3

EXPORTS = [
    "cc_init", "cc_shutdown", "cc_last_cuda_error", "cc_kernel_launches", "cc_workspace_bytes",
    "cc_register_region", "cc_unregister_region", "cc_log_attach", "cc_log_reset", "cc_log_reset_async", "cc_log_mirror_attach", "cc_log_drain", "cc_log_drain_start", "cc_log_drain_wait", "cc_log_drain_stop",
    "cc_checkpoint_ex", "cc_checkpoint_delta", "cc_checkpoint_delta_fused", "cc_checkpoint_delta_rle", "cc_checkpoint_marked", "cc_checkpoint_versions",
    "cc_checkpoint_all", "cc_checkpoint_all_rle", "cc_snapshot_region", "cc_compact_log", "cc_scan_only", "cc_trace_events", "cc_dirty_list", "cc_apply_scratch_bytes", "cc_apply_attach", "cc_apply_stage_attach", "cc_apply_stage_stats", "cc_apply_log",
    "cc_worker_start", "cc_worker_stop", "cc_worker_alive", "cc_worker_footprint", "cc_peek_queue", "cc_submit", "cc_measure_submit_cost", "cc_measure_launch_cost", "cc_poll", "cc_wait",
    "cc_dirty_pages_static",
]


class cc_config(ctypes.Structure):
    _fields_ = [("ring_capacity", ctypes.c_uint32), ("worker_blocks", ctypes.c_uint32),
                ("worker_threads", ctypes.c_uint32), ("backoff_ns", ctypes.c_uint32),
                ("max_lifetime_ns", ctypes.c_uint64)]


class cc_region_desc(ctypes.Structure):
    _fields_ = [("region_id", ctypes.c_uint32), ("page_bytes", ctypes.c_uint32), ("bytes", ctypes.c_uint64),
                ("base", ctypes.c_void_p), ("shadow", ctypes.c_void_p), ("workspace", ctypes.c_void_p),
                ("workspace_bytes", ctypes.c_uint64), ("flags", ctypes.c_uint32), ("reserved", ctypes.c_uint32)]


class cc_ckpt_opts(ctypes.Structure):
    _fields_ = [("discovery", ctypes.c_uint32), ("path", ctypes.c_uint32), ("run_pages", ctypes.c_uint32),
                ("mark_flags", ctypes.c_uint32), ("dirty_bitmap", ctypes.c_void_p), ("version", ctypes.c_void_p),
                ("committed", ctypes.c_void_p)]


class cc_result(ctypes.Structure):
    _fields_ = [("seq_done", ctypes.c_uint64), ("n_dirty", ctypes.c_uint64), ("bytes", ctypes.c_uint64),
                ("log_offset_after", ctypes.c_uint64), ("epoch", ctypes.c_uint64), ("status", ctypes.c_int32),
                ("flags", ctypes.c_uint32), ("t_start_ns", ctypes.c_uint64), ("t_end_ns", ctypes.c_uint64)]

    def as_dict(self):
        return {f: getattr(self, f) for f, _ in self._fields_}


class cc_task(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_uint32), ("region_id", ctypes.c_uint32), ("flags", ctypes.c_uint32),
                ("version", ctypes.c_uint32), ("seq", ctypes.c_uint64), ("epoch", ctypes.c_uint64),
                ("arg0", ctypes.c_uint64), ("arg1", ctypes.c_uint64), ("arg2", ctypes.c_uint64),
                ("arg3", ctypes.c_uint64)]


assert ctypes.sizeof(cc_result) == 64 and ctypes.sizeof(cc_task) == 64

_lib = None


def lib_path() -> str:
    return _build.LIB


def load_library():
    """dlopen libconcordia.so (building it if the sources are newer) and declare the signatures."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    lib = ctypes.CDLL(path)
    vp, u32, u64, i32 = ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int32
    P = ctypes.POINTER
    sig = {
        "cc_init": (i32, [P(vp), i32, P(cc_config)]),
        "cc_shutdown": (i32, [vp]),
        "cc_last_cuda_error": (i32, [vp]),
        "cc_kernel_launches": (u64, [vp]),
        "cc_workspace_bytes": (u64, [u64, u32]),
        "cc_register_region": (i32, [vp, P(cc_region_desc)]),
        "cc_unregister_region": (i32, [vp, u32]),
        "cc_log_attach": (i32, [vp, vp, u64, vp]),
        "cc_log_reset": (i32, [vp]),
        "cc_log_reset_async": (i32, [vp, vp]),
        "cc_log_mirror_attach": (i32, [vp, vp, u64, vp]),
        "cc_log_drain": (i32, [vp, u64, vp, vp]),
        "cc_log_drain_start": (i32, [vp]),
        "cc_log_drain_wait": (i32, [vp, u64, u64]),
        "cc_log_drain_stop": (i32, [vp]),
        "cc_checkpoint_ex": (i32, [vp, u32, u64, P(cc_ckpt_opts), vp, vp]),
        "cc_checkpoint_delta": (i32, [vp, u32, u64, vp, vp]),
        "cc_checkpoint_delta_fused": (i32, [vp, u32, u64, vp, vp]),
        "cc_checkpoint_delta_rle": (i32, [vp, u32, u64, u32, vp, vp]),
        "cc_checkpoint_marked": (i32, [vp, u32, u64, vp, u32, vp, vp]),
        "cc_checkpoint_versions": (i32, [vp, u32, u64, vp, vp, vp, vp]),
        "cc_checkpoint_all": (i32, [vp, u64, vp, vp]),
        "cc_checkpoint_all_rle": (i32, [vp, u64, u32, vp, vp]),
        "cc_snapshot_region": (i32, [vp, u32, u64, vp, vp]),
        "cc_compact_log": (i32, [vp, vp, u64, vp, u64, vp, vp]),
        "cc_scan_only": (i32, [vp, u32, vp, vp]),
        "cc_trace_events": (i32, [vp, vp, vp]),
        "cc_dirty_list": (i32, [vp, u32, P(vp), P(vp)]),
        "cc_apply_scratch_bytes": (u64, [u64]),
        "cc_apply_attach": (i32, [vp, vp, u64]),
        "cc_apply_stage_attach": (i32, [vp, vp, u64]),
        "cc_apply_stage_stats": (i32, [vp, P(u64), P(u64)]),
        "cc_apply_log": (i32, [vp, vp, u64, vp, vp]),
        "cc_worker_start": (i32, [vp]),
        "cc_worker_stop": (i32, [vp]),
        "cc_worker_alive": (i32, [vp]),
        "cc_worker_footprint": (i32, [vp, P(u32), P(u32), P(u32), P(u32), P(u32)]),
        "cc_peek_queue": (i32, [vp, P(u64), P(u64)]),
        "cc_submit": (i32, [vp, P(cc_task), P(u64)]),
        "cc_measure_submit_cost": (i32, [vp, u32, P(ctypes.c_double)]),
        "cc_measure_launch_cost": (i32, [vp, u32, vp, P(ctypes.c_double), P(ctypes.c_double)]),
        "cc_poll": (i32, [vp, u64, P(cc_result)]),
        "cc_wait": (i32, [vp, u64, u64, P(cc_result)]),
        "cc_dirty_pages_static": (i32, [i32, vp, vp, u64, u32, vp, u32, vp, vp, P(i32)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


class ConcordiaError(RuntimeError):
    def __init__(self, call, code, cuda=0):
        super().__init__("%s failed: status %d (cuda error %d)" % (call, code, cuda))
        self.code = code


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def dirty_pages_static(cur: torch.Tensor, shadow: torch.Tensor, page_bytes: int, d_list: torch.Tensor,
                       d_count: torch.Tensor, stream=None):
    """cc_dirty_pages_static: the ascending dirty page list of `cur` against `shadow` for callers that cannot
    allocate -- no Context, no registered region, no workspace; the scratch is a fixed array inside the library
    (at most CC_STATIC_MAX_PAGES pages, else ConcordiaError with code CC_ERR_STATIC_LIMIT).  Every tensor is the
    caller's: cur / shadow contiguous CUDA tensors of equal byte size, d_list an int32 CUDA tensor that receives
    min(k, d_list.numel()) page indices, d_count an int32 CUDA (or pinned) tensor of one element that receives
    k.  Asynchronous on `stream` (default: torch's current stream).  Calls that can overlap on one GPU race on the
    shared scratch; the first call on a device does the one-time set-up and belongs outside stream capture.
    This wrapper marshals arguments and allocates no device memory either."""
    assert cur.is_cuda and cur.is_contiguous() and shadow.is_cuda and shadow.is_contiguous()
    nbytes = cur.numel() * cur.element_size()
    assert shadow.numel() * shadow.element_size() == nbytes and shadow.device == cur.device
    assert d_list.dtype == torch.int32 and d_list.is_cuda and d_list.is_contiguous()
    assert d_count.dtype == torch.int32 and d_count.numel() == 1 and (d_count.is_cuda or d_count.is_pinned())
    lib = load_library()
    err = ctypes.c_int32(0)
    if stream is None:
        stream = torch.cuda.current_stream(cur.device)
    rc = lib.cc_dirty_pages_static(cur.device.index, cur.data_ptr(), shadow.data_ptr(), nbytes, page_bytes,
                                   d_list.data_ptr() if d_list.numel() else None, d_list.numel(), d_count.data_ptr(),
                                   ctypes.c_void_p(stream.cuda_stream), ctypes.byref(err))
    if rc != CC_OK:
        raise ConcordiaError("cc_dirty_pages_static", rc, err.value)


class Result:
    """A 64-byte cc_result in pinned host memory that the GPU writes."""

    def __init__(self):
        self.buf = torch.zeros(64, dtype=torch.uint8, pin_memory=True)
        self.ptr = self.buf.data_ptr()

    def clear(self):
        self.buf.zero_()

    def read(self) -> cc_result:
        return cc_result.from_buffer_copy(self.buf.numpy().tobytes())


class Context:
    """One libconcordia context on one CUDA device.  Same names as the C ABI, minus the cc_ prefix."""

    def __init__(self, device: int = 0, ring_capacity: int = 0, worker_blocks: int = 0, worker_threads: int = 0,
                 backoff_ns: int = 0, max_lifetime_ns: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_23521_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.lib = load_library()
        self.device = device
        cfg = cc_config(ring_capacity, worker_blocks, worker_threads, backoff_ns, max_lifetime_ns)
        h = ctypes.c_void_p()
        rc = self.lib.cc_init(ctypes.byref(h), device, ctypes.byref(cfg))
        if rc != CC_OK:
            raise ConcordiaError("cc_init", rc)
        self.h = h
        self._keep = {}     # region_id -> tensors we must keep alive
        self._log = None
        self._committed = None
        self._scratch = None
        self._stage = None
        self._mirror = None

    # -- helpers
    def _check(self, call, rc):
        if rc < 0:
            raise ConcordiaError(call, rc, self.lib.cc_last_cuda_error(self.h))
        return rc

    def kernel_launches(self) -> int:
        return int(self.lib.cc_kernel_launches(self.h))

    def workspace_bytes(self, nbytes: int, page_bytes: int) -> int:
        return int(self.lib.cc_workspace_bytes(nbytes, page_bytes))

    # -- regions
    def register_region(self, region_id: int, base: torch.Tensor, page_bytes: int, shadow: torch.Tensor = None,
                        snapshot_now: bool = True, no_shadow: bool = False):
        """base/shadow: contiguous CUDA tensors of equal byte size.  Allocates shadow and workspace with
        torch if not given.  Returns the shadow tensor (uint8 view), or None for an allocator-aware
        region registered with no_shadow=True (CC_REG_NO_SHADOW)."""
        assert base.is_cuda and base.is_contiguous()
        nbytes = base.numel() * base.element_size()
        if no_shadow:
            assert shadow is None
            snapshot_now = False
        elif shadow is None:
            shadow = torch.empty(nbytes, dtype=torch.uint8, device=base.device)
        assert no_shadow or (shadow.is_cuda and shadow.is_contiguous() and shadow.numel() * shadow.element_size() == nbytes)
        wsb = self.workspace_bytes(nbytes, page_bytes)
        if wsb == 0:
            raise ConcordiaError("cc_workspace_bytes", CC_ERR_INVALID)
        ws = torch.empty(wsb + 256, dtype=torch.uint8, device=base.device)
        off = (-ws.data_ptr()) % 256
        flags = (CC_REG_SNAPSHOT_NOW if snapshot_now else 0) | (CC_REG_NO_SHADOW if no_shadow else 0)
        d = cc_region_desc(region_id, page_bytes, nbytes, base.data_ptr(), None if no_shadow else shadow.data_ptr(),
                           ws.data_ptr() + off, wsb, flags, 0)
        self._check("cc_register_region", self.lib.cc_register_region(self.h, ctypes.byref(d)))
        self._keep[region_id] = (base, shadow, ws)
        return shadow

    def unregister_region(self, region_id: int):
        self._check("cc_unregister_region", self.lib.cc_unregister_region(self.h, region_id))
        self._keep.pop(region_id, None)

    # -- log
    def log_attach(self, log: torch.Tensor, committed_off: torch.Tensor = None):
        """log: uint8 tensor, CUDA or pinned host.  committed_off: pinned int64[1] (optional)."""
        assert log.dtype == torch.uint8 and log.is_contiguous() and (log.is_cuda or log.is_pinned())
        cptr = None
        if committed_off is not None:
            assert committed_off.numel() * committed_off.element_size() >= 8
            cptr = ctypes.c_void_p(committed_off.data_ptr())
        self._check("cc_log_attach", self.lib.cc_log_attach(self.h, log.data_ptr(), log.numel(), cptr))
        self._log, self._committed = log, committed_off

    def log_mirror_attach(self, host_log: torch.Tensor, committed_off: torch.Tensor = None):
        """host_log: pinned uint8 tensor mirroring the (device-resident) attached log; None detaches."""
        if host_log is None:
            self._check("cc_log_mirror_attach", self.lib.cc_log_mirror_attach(self.h, None, 0, None))
            self._mirror = None
            return
        assert host_log.dtype == torch.uint8 and host_log.is_contiguous() and host_log.is_pinned()
        cptr = ctypes.c_void_p(committed_off.data_ptr()) if committed_off is not None else None
        self._check("cc_log_mirror_attach", self.lib.cc_log_mirror_attach(self.h, host_log.data_ptr(), host_log.numel(), cptr))
        self._mirror = (host_log, committed_off)

    def log_drain(self, upto: int, copy_stream, after_stream=None):
        self._check("cc_log_drain", self.lib.cc_log_drain(self.h, upto, _stream_ptr(after_stream), _stream_ptr(copy_stream)))

    def log_drain_start(self):
        """Start the library's drainer thread (device log -> attached host mirror, copy engine, no per-step call)."""
        self._check("cc_log_drain_start", self.lib.cc_log_drain_start(self.h))

    def log_drain_wait(self, upto: int, timeout_s: float = 30.0):
        self._check("cc_log_drain_wait", self.lib.cc_log_drain_wait(self.h, upto, int(timeout_s * 1e9)))

    def log_drain_stop(self):
        self._check("cc_log_drain_stop", self.lib.cc_log_drain_stop(self.h))

    def log_reset(self):
        self._check("cc_log_reset", self.lib.cc_log_reset(self.h))

    def log_reset_async(self, stream=None):
        self._check("cc_log_reset_async", self.lib.cc_log_reset_async(self.h, _stream_ptr(stream)))

    # -- host-launched path
    def checkpoint_delta(self, region_id: int, epoch: int, result: Result = None, stream=None):
        self._check("cc_checkpoint_delta", self.lib.cc_checkpoint_delta(
            self.h, region_id, epoch, _stream_ptr(stream), ctypes.c_void_p(result.ptr) if result else None))

    def checkpoint_ex(self, region_id: int, epoch: int, result: Result = None, stream=None, discovery: int = CC_DISC_SCAN,
                      path: int = CC_PATH_AUTO, run_pages: int = 0, dirty_bitmap: torch.Tensor = None, mark_flags: int = 0,
                      version: torch.Tensor = None, committed: torch.Tensor = None):
        """The general checkpoint call (cc_checkpoint_ex): discovery x record kind x path."""
        o = cc_ckpt_opts(discovery, path, run_pages, mark_flags,
                         dirty_bitmap.data_ptr() if dirty_bitmap is not None else None,
                         version.data_ptr() if version is not None else None,
                         committed.data_ptr() if committed is not None else None)
        self._check("cc_checkpoint_ex", self.lib.cc_checkpoint_ex(
            self.h, region_id, epoch, ctypes.byref(o), _stream_ptr(stream), ctypes.c_void_p(result.ptr) if result else None))

    def checkpoint_delta_fused(self, region_id: int, epoch: int, result: Result = None, stream=None):
        self._check("cc_checkpoint_delta_fused", self.lib.cc_checkpoint_delta_fused(
            self.h, region_id, epoch, _stream_ptr(stream), ctypes.c_void_p(result.ptr) if result else None))

    def checkpoint_delta_rle(self, region_id: int, epoch: int, run_pages: int, result: Result = None, stream=None):
        self._check("cc_checkpoint_delta_rle", self.lib.cc_checkpoint_delta_rle(
            self.h, region_id, epoch, run_pages, _stream_ptr(stream), ctypes.c_void_p(result.ptr) if result else None))

    def checkpoint_marked(self, region_id: int, epoch: int, dirty_bitmap: torch.Tensor, flags: int = 0,
                          result: Result = None, stream=None):
        """dirty_bitmap: CUDA int32/uint32 tensor of ceil(n_pages/32) words (bit p&31 of word p>>5)."""
        assert dirty_bitmap.is_cuda and dirty_bitmap.is_contiguous() and dirty_bitmap.element_size() == 4
        self._check("cc_checkpoint_marked", self.lib.cc_checkpoint_marked(
            self.h, region_id, epoch, dirty_bitmap.data_ptr(), flags, _stream_ptr(stream),
            ctypes.c_void_p(result.ptr) if result else None))

    def checkpoint_versions(self, region_id: int, epoch: int, version: torch.Tensor, committed: torch.Tensor,
                            result: Result = None, stream=None):
        """version / committed: CUDA int64 tensors with one entry per page; committed is advanced in place."""
        for t in (version, committed):
            assert t.is_cuda and t.is_contiguous() and t.element_size() == 8
        self._check("cc_checkpoint_versions", self.lib.cc_checkpoint_versions(
            self.h, region_id, epoch, version.data_ptr(), committed.data_ptr(), _stream_ptr(stream),
            ctypes.c_void_p(result.ptr) if result else None))

    def checkpoint_all(self, epoch: int, result: Result = None, stream=None):
        self._check("cc_checkpoint_all", self.lib.cc_checkpoint_all(
            self.h, epoch, _stream_ptr(stream), ctypes.c_void_p(result.ptr) if result else None))

    def checkpoint_all_rle(self, epoch: int, run_pages: int, result: Result = None, stream=None):
        self._check("cc_checkpoint_all_rle", self.lib.cc_checkpoint_all_rle(
            self.h, epoch, run_pages, _stream_ptr(stream), ctypes.c_void_p(result.ptr) if result else None))

    def snapshot_region(self, region_id: int, epoch: int, result: Result = None, stream=None):
        self._check("cc_snapshot_region", self.lib.cc_snapshot_region(
            self.h, region_id, epoch, _stream_ptr(stream), ctypes.c_void_p(result.ptr) if result else None))

    def compact_log(self, in_log: torch.Tensor, in_bytes: int, out_log: torch.Tensor, result: Result = None, stream=None):
        for t in (in_log, out_log):
            assert t.dtype == torch.uint8 and t.is_contiguous() and (t.is_cuda or t.is_pinned())
        assert in_bytes <= in_log.numel()
        self._check("cc_compact_log", self.lib.cc_compact_log(
            self.h, in_log.data_ptr(), in_bytes, out_log.data_ptr(), out_log.numel(), _stream_ptr(stream),
            ctypes.c_void_p(result.ptr) if result else None))

    def scan_only(self, region_id: int, result: Result = None, stream=None):
        self._check("cc_scan_only", self.lib.cc_scan_only(
            self.h, region_id, _stream_ptr(stream), ctypes.c_void_p(result.ptr) if result else None))

    def trace_events(self, after_scan: "torch.cuda.Event" = None, after_compact: "torch.cuda.Event" = None):
        """Events (created with enable_timing=True and recorded once, so that the handle exists) that the
        next host-launched calls record after the scan / compaction kernels; None switches it off."""
        a = ctypes.c_void_p(after_scan.cuda_event) if after_scan is not None else None
        b = ctypes.c_void_p(after_compact.cuda_event) if after_compact is not None else None
        self._check("cc_trace_events", self.lib.cc_trace_events(self.h, a, b))

    def dirty_list(self, region_id: int) -> torch.Tensor:
        """Ascending dirty page indices of the last scan as an int64 CPU tensor (synchronises)."""
        dl, dc = ctypes.c_void_p(), ctypes.c_void_p()
        self._check("cc_dirty_list", self.lib.cc_dirty_list(self.h, region_id, ctypes.byref(dl), ctypes.byref(dc)))
        base, _, ws = self._keep[region_id]
        torch.cuda.current_stream().synchronize()
        ws_off = dc.value - ws.data_ptr()
        k = int(ws[ws_off:ws_off + 4].view(torch.int32).item())
        d_off = dl.value - ws.data_ptr()
        return ws[d_off:d_off + 4 * k].view(torch.int32).to(torch.int64).cpu()

    def apply_attach(self, max_records: int, device=None):
        nb = int(self.lib.cc_apply_scratch_bytes(max_records))
        if nb == 0:
            raise ConcordiaError("cc_apply_scratch_bytes", CC_ERR_INVALID)
        s = torch.empty(nb + 256, dtype=torch.uint8, device=device or torch.device("cuda", self.device))
        off = (-s.data_ptr()) % 256
        self._check("cc_apply_attach", self.lib.cc_apply_attach(self.h, s.data_ptr() + off, nb))
        self._scratch = s

    def apply_stage_attach(self, nbytes: int):
        """Allocate and attach a device staging buffer for host-resident logs (0 detaches)."""
        if nbytes == 0:
            self._check("cc_apply_stage_attach", self.lib.cc_apply_stage_attach(self.h, None, 0))
            self._stage = None
            return
        s = torch.empty(nbytes + 16, dtype=torch.uint8, device=torch.device("cuda", self.device))
        off = (-s.data_ptr()) % 16
        self._check("cc_apply_stage_attach", self.lib.cc_apply_stage_attach(self.h, s.data_ptr() + off, nbytes))
        self._stage = s

    def apply_stage_stats(self):
        """(staged, bypassed): host-resident logs copied into the staging buffer / read in place although one is attached."""
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        self._check("cc_apply_stage_stats", self.lib.cc_apply_stage_stats(self.h, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def apply_log(self, log: torch.Tensor, nbytes: int, result: Result = None, stream=None):
        assert log.dtype == torch.uint8 and log.is_contiguous() and (log.is_cuda or log.is_pinned())
        assert nbytes <= log.numel()
        self._check("cc_apply_log", self.lib.cc_apply_log(
            self.h, log.data_ptr(), nbytes, _stream_ptr(stream), ctypes.c_void_p(result.ptr) if result else None))

    # -- ring + persistent worker
    def worker_start(self):
        # everything the worker touches is allocated; make sure nothing of ours is still queued
        torch.cuda.synchronize(self.device)
        self._check("cc_worker_start", self.lib.cc_worker_start(self.h))

    def worker_stop(self):
        self._check("cc_worker_stop", self.lib.cc_worker_stop(self.h))

    def worker_alive(self) -> bool:
        return self.lib.cc_worker_alive(self.h) == 1

    def worker_footprint(self) -> dict:
        v = [ctypes.c_uint32() for _ in range(5)]
        self._check("cc_worker_footprint", self.lib.cc_worker_footprint(self.h, *[ctypes.byref(x) for x in v]))
        b, t, sm, rg, sms = [x.value for x in v]
        # CTAs of this shape one SM holds (B200: 64 Ki registers, 2,048 threads, 227 KiB of shared memory + 1 KiB reserved per CTA);
        # the worker's share of the GPU = its CTAs / the CTA slots of the whole device
        fit = max(1, min(65536 // max(1, rg * t), 2048 // max(1, t), (227 * 1024) // (sm + 1024)))
        return {"blocks": b, "threads_per_block": t, "smem_bytes_per_block": sm, "registers_per_thread": rg, "sm_count": sms,
                "blocks_that_fit_per_sm": fit, "sm_share_pct": round(100.0 * min(b, sms * fit) / (sms * fit), 2)}

    def peek_queue(self):
        h, t = ctypes.c_uint64(), ctypes.c_uint64()
        self._check("cc_peek_queue", self.lib.cc_peek_queue(self.h, ctypes.byref(h), ctypes.byref(t)))
        return h.value, t.value

    def submit(self, kind: int, region_id: int = 0, epoch: int = 0, arg0: int = 0, arg1: int = 0, arg2: int = 0,
               arg3: int = 0, flags: int = 0) -> int:
        """Returns the sequence number, or raises ConcordiaError(CC_ERR_RING_FULL)."""
        t = cc_task(kind, region_id, flags, 0, 0, epoch, arg0, arg1, arg2, arg3)
        seq = ctypes.c_uint64()
        self._check("cc_submit", self.lib.cc_submit(self.h, ctypes.byref(t), ctypes.byref(seq)))
        return seq.value

    def measure_submit_cost(self, n: int = 100000) -> float:
        """Mean host cost of cc_submit in ns, measured inside the library (no ctypes in the timed section)."""
        v = ctypes.c_double()
        self._check("cc_measure_submit_cost", self.lib.cc_measure_submit_cost(self.h, n, ctypes.byref(v)))
        return v.value

    def measure_launch_cost(self, n: int = 2000, stream=None):
        """(ns per empty-kernel launch with a sync each, ns per launch when batched) -- PAPER.md Table 7."""
        a, b = ctypes.c_double(), ctypes.c_double()
        self._check("cc_measure_launch_cost", self.lib.cc_measure_launch_cost(self.h, n, _stream_ptr(stream), ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def poll(self, seq: int):
        r = cc_result()
        rc = self._check("cc_poll", self.lib.cc_poll(self.h, seq, ctypes.byref(r)))
        return None if rc == CC_PENDING else r

    def wait(self, seq: int, timeout_s: float = 10.0) -> cc_result:
        r = cc_result()
        self._check("cc_wait", self.lib.cc_wait(self.h, seq, int(timeout_s * 1e9), ctypes.byref(r)))
        return r

    def shutdown(self):
        if self.h:
            rc = self.lib.cc_shutdown(self.h)
            self.h = None
            self._keep.clear()
            if rc < 0:
                raise ConcordiaError("cc_shutdown", rc)

    def __del__(self):
        try:
            self.shutdown()
        except Exception:
            pass
