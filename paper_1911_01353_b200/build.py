"""Build the C-ABI shared library (CUDA, sm_100a only) in-tree: paper_1911_01353_b200/libjerk_b200.so."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "csrc", "jerk.cu"), os.path.join(HERE, "csrc", "jerk_spectrum.cu")]
DEPS = SRCS + [os.path.join(HERE, "csrc", "jerk_fft.cuh"), os.path.join(HERE, "csrc", "jerk_fft64.cuh"),
               os.path.join(os.path.dirname(HERE), "include", "jerk.h")]
LIB = os.path.join(HERE, "libjerk_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu into libjerk_b200.so (skipped when the library is newer than every source)."""
    if not force and not needs_build():
        return LIB
    target = LIB
    cmd = [nvcc_path()] + NVCC_FLAGS + ["-o", target] + SRCS
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libjerk_b200.so")
    return target


if __name__ == "__main__":
    print(build(force=True, verbose=True))
