"""Build libcdmt.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcdmt.so")
SOURCES = ["cdmt_kernels.cu", "cdmt_fused.cu", "cdmt_fused2.cu", "cdmt_fused4.cu", "cdmt_fused5.cu", "cdmt_redigitize.cu", "cdmt_incoherent.cu", "cdmt_api.cu"]
HEADERS = ["cdmt_fft.cuh", "cdmt_fft2.cuh", "cdmt_tmem.cuh", "cdmt_fused_common.cuh", "cdmt_internal.h", os.path.join("..", "..", "include", "cdmt.h")]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "--threads", "4"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    for f in SOURCES + HEADERS:
        if os.path.getmtime(os.path.join(CSRC, f)) > t:
            return True
    return False


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        objs = []
        procs = []
        for src in SOURCES:
            obj = os.path.join(CSRC, src.replace(".cu", ".o"))
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
                  ["-c", os.path.join(CSRC, src), "-o", obj]
            procs.append((subprocess.Popen(cmd), cmd))
            objs.append(obj)
        for pr, cmd in procs:
            if pr.wait() != 0:
                raise RuntimeError("nvcc failed: " + " ".join(cmd))
        tmp = LIB + ".tmp%d" % os.getpid()
        subprocess.check_call([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
