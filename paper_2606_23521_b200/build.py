"""Build libconcordia.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libconcordia.so")
SOURCES = ["concordia.cu", "cc_static.cu"]
HEADERS = ["cc_common.cuh", "cc_crc.cuh", "cc_ckpt.cuh", "cc_mark.cuh", "cc_fused.cuh", "cc_pass.cuh", "cc_small.cuh", "cc_tasks.cuh", "cc_rle.cuh", "cc_apply.cuh",
           "cc_apply_parse.cuh", "cc_compactor.cuh", "cc_batch.cuh", "cc_worker.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    deps.append(os.path.join(os.path.dirname(_HERE), "include", "concordia.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + ".tmp.%d" % os.getpid()
        extra = os.environ.get("CC_NVCC_FLAGS", "").split()         # e.g. -DCC_LD_NC=1 for an A/B build
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + \
              [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
