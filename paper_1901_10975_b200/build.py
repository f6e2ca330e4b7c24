"""Build libcn.so in-tree with nvcc for sm_100a (no torch, no JIT cache)."""
from __future__ import annotations

import os
import subprocess
from pathlib import Path

HERE = Path(__file__).resolve().parent
SO = HERE / "libcn.so"
SRCS = [HERE / "csrc" / "cn_api.cu"]
DEPS = SRCS + [HERE / "csrc" / "cn_device.cuh", HERE / "csrc" / "cn_tape.cuh",
               HERE / "csrc" / "cn_host.hpp", HERE / "csrc" / "cn_layout.hpp",
               HERE / "csrc" / "cn_finalize.hpp",
               HERE / "csrc" / "cn_tape_program.hpp",
               HERE.parent / "include" / "cn.h"]

NVCC_FLAGS = (["-DCN_TRACE"] if os.environ.get("CN_TRACE") else []) + ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-pthread", "-shared"]


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and SO.exists() and SO.stat().st_mtime >= max(p.stat().st_mtime for p in DEPS):
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = SO.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
        ["-o", str(tmp)] + [str(s) for s in SRCS]
    subprocess.check_call(cmd)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force=True, verbose=True))
