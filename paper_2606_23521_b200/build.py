"""Build libconcordia.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libconcordia.so")
SOURCES = ["concordia.cu"]
HEADERS = ["cc_common.cuh", "cc_crc.cuh", "cc_ckpt.cuh", "cc_mark.cuh", "cc_fused.cuh", "cc_rle.cuh", "cc_apply.cuh", "cc_compactor.cuh", "cc_batch.cuh", "cc_worker.cuh"]
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
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + \
              [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


PROBES = ["link_probe.cu", "scan_probe.cu"]        # standalone measurement programs (profiles/r01_*_probe.md)


def build_probes(force: bool = False) -> list:
    """Compile the standalone measurement programs into paper_2606_23521_b200/bin/ (git-ignored)."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    out_dir = os.path.join(_HERE, "bin")
    os.makedirs(out_dir, exist_ok=True)
    outs = []
    for src in PROBES:
        s = os.path.join(CSRC, src)
        o = os.path.join(out_dir, src[:-3])
        if force or not os.path.exists(o) or os.path.getmtime(o) < os.path.getmtime(s):
            subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-o", o, s], check=True)
        outs.append(o)
    return outs


if __name__ == "__main__":
    print(build(force=True, verbose=True))
