import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(autouse=True)
def _release_cached_device_memory(request):
    """The full-size GPU tests skip themselves when free device memory is short; give back what earlier tests'
    tensors left in torch's caching allocator first, so that a skip means the box is too small, not the cache full."""
    if "gpu" in request.keywords:
        import gc
        import torch
        gc.collect()
        if torch.cuda.is_available():
            torch.cuda.empty_cache()
    yield


# ---- every checkpoint path under the same parity tests ----
# cc_checkpoint_delta & co. choose between the single-pass kernel and the classic phases by region size and log
# placement (CC_PATH_AUTO).  The small-shape parity modules below run three times: as written (auto), with every
# checkpoint call forced onto the phases, and forced onto the single pass -- the bytes must not depend on the path.
PATH_MODULES = {"test_gpu_checkpoint", "test_gpu_marked", "test_gpu_rle", "test_gpu_fused", "test_gpu_history", "test_gpu_compact"}


def pytest_generate_tests(metafunc):
    if metafunc.module.__name__ in PATH_MODULES and "ckpt_path" not in metafunc.fixturenames:
        metafunc.fixturenames.append("ckpt_path")
        metafunc.parametrize("ckpt_path", ["auto", "phases", "single"], indirect=True)


@pytest.fixture
def ckpt_path(request, monkeypatch):
    mode = getattr(request, "param", "auto")
    if mode == "auto":
        return mode
    import paper_2606_23521_b200 as cc
    C = cc.Context
    forced = cc.CC_PATH_PHASES if mode == "phases" else cc.CC_PATH_SINGLE_PASS

    def path_for(run_pages):
        if forced == cc.CC_PATH_SINGLE_PASS and run_pages > 32:
            return cc.CC_PATH_PHASES            # the single pass takes run_pages <= 32
        return forced

    monkeypatch.setattr(C, "checkpoint_delta", lambda self, rid, epoch, result=None, stream=None:
                        C.checkpoint_ex(self, rid, epoch, result, stream, path=forced))
    monkeypatch.setattr(C, "checkpoint_delta_rle", lambda self, rid, epoch, run_pages, result=None, stream=None:
                        C.checkpoint_ex(self, rid, epoch, result, stream, path=path_for(run_pages), run_pages=run_pages)
                        if run_pages else C.checkpoint_ex(self, rid, epoch, result, stream, run_pages=0xFFFFFFFF))
    monkeypatch.setattr(C, "checkpoint_marked", lambda self, rid, epoch, bm, flags=0, result=None, stream=None:
                        C.checkpoint_ex(self, rid, epoch, result, stream, discovery=cc.CC_DISC_MARKS, path=forced,
                                        dirty_bitmap=bm, mark_flags=flags))
    monkeypatch.setattr(C, "checkpoint_versions", lambda self, rid, epoch, v, c, result=None, stream=None:
                        C.checkpoint_ex(self, rid, epoch, result, stream, discovery=cc.CC_DISC_VERSIONS, path=forced, version=v, committed=c))
    monkeypatch.setattr(C, "snapshot_region", lambda self, rid, epoch, result=None, stream=None:
                        C.checkpoint_ex(self, rid, epoch, result, stream, discovery=cc.CC_DISC_ALL, path=forced))
    return mode
