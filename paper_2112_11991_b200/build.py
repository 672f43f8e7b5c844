"""Build libtb.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2112_11991_b200.build [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB_DIR = os.path.join(HERE, "lib")
LIB_PATH = os.path.join(LIB_DIR, "libtb.so")
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")
SOURCES = ["tb_api.cu", "tb_bank.cu", "tb_noalloc.cu"]
DEPS = ["tb_api.cu", "tb_bank.cu", "tb_noalloc.cu", "tb_kernels.cuh", "tb_fft.cuh", "tb_reduce.cuh", "tb_whiten.cuh", os.path.join("..", "..", "include", "tb.h")]


def needs_build() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(verbose: bool = False, force: bool = False) -> str:
    if not force and not needs_build():
        return LIB_PATH
    os.makedirs(LIB_DIR, exist_ok=True)
    nvcc = os.path.join(CUDA_HOME, "bin", "nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
           "-o", LIB_PATH] + [os.path.join(CSRC, s) for s in SOURCES] + \
          ["-lcufft", f"-L{CUDA_HOME}/lib64", "-Xlinker", f"-rpath={CUDA_HOME}/lib64"]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stderr)
    return LIB_PATH


if __name__ == "__main__":
    print(build(verbose="--verbose" in sys.argv, force=True))
