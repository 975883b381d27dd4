"""Build libspt.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2606_27262_b200.build [--force]

nvcc cross-compiles without a GPU, so this also is the "does it build" check on the CPU box.
"""
from __future__ import annotations

import fcntl
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libspt.so")
SOURCES = ["api.cu", "plan.cpp", "dedisperse.cu", "sps.cu", "peaks.cu", "peaks_static.cu", "stream.cu", "sift.cu", "cutout.cu", "probe.cu"]
HEADERS = ["internal.h", "kernels.h", os.path.join("..", "..", "include", "spt.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--fmad=false",
         "-Xcompiler", "-fPIC,-ffp-contract=off,-O2,-pthread", "-Xptxas", "-v", "-shared", "-cudart", "static"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    # several ranks of one node may get here together (torchrun): one builds, the others wait on the lock and find the
    # library fresh; the library appears under its name only when complete (rename)
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not _stale():
                return LIB
            tmp = LIB + ".tmp.%d" % os.getpid()
            extra = os.environ.get("SPT_NVCC_EXTRA", "").split()      # e.g. -DSPS_ITERS=9 for an A/B build
            cmd = [NVCC, *FLAGS, *extra, "-o", tmp, *[os.path.join(CSRC, s) for s in SOURCES]]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if verbose or r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode != 0:
                if os.path.exists(tmp):
                    os.unlink(tmp)
                raise RuntimeError("nvcc failed building libspt.so")
            os.replace(tmp, LIB)
            with open(os.path.join(HERE, "build.log"), "w") as f:
                f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
