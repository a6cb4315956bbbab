"""Build libemu4pi.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libemu4pi.so")
SOURCES = ["emu_api.cu", "emu_bin.cu", "emu_find.cu", "emu_fit.cu", "emu_recognize.cu"]
HEADERS = ["emu_dev.cuh", "emu_host.h", os.path.join("..", "..", "include", "emu.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        if not os.path.exists(nvcc):
            nvcc = "nvcc"
        extra = os.environ.get("EMU_NVCC_EXTRA", "").split()       # tuning experiments only (e.g. -DEMU_REFILL=12)
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
        subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB


def build_microbench(out_dir: str) -> str:
    """Compile the stand-alone issue-rate micro-benchmark (microbench/mb_pipes.cu: the measured peak of the voting
    kernel's instruction mix) into `out_dir` and return the executable's path.  Not part of the library
    and not built by build(): bench.py runs it as a leg of its own, a CPU test checks that it compiles."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc):
        nvcc = "nvcc"
    exe = os.path.join(out_dir, "mb_pipes")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe,
                    os.path.join(HERE, "microbench", "mb_pipes.cu")], check=True)
    return exe


if __name__ == "__main__":
    print(build(force=True, verbose=True))
