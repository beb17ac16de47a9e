"""Build the C-ABI library ``libnasg_b200.so`` for sm_100a with nvcc (cross-compiles without a GPU).

    python -m paper_2606_09794_b200.build [--force] [--verbose]

The .so is written next to this file (in-tree, git-ignored) so that it travels to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SOURCES = [os.path.join(CSRC, f) for f in ("nasg_api.cu", "nasg_kernels.cu", "nasg_pipe_kernels.cu", "nasg_tile_kernels.cu", "nasg_rec_kernels.cu", "sh_kernels.cu",
                                               "sh_pipe_kernels.cu", "nasg_host_pipeline.cu", "nasg_noalloc.cu", "nasg_rec_convert.cu")]
HEADERS = [os.path.join(CSRC, f) for f in ("nasg_internal.h", "nasg_math.cuh", "nasg_lp_math.cuh", "bulk_common.cuh", "pipe_common.cuh", "sh_math.cuh")] + [
    os.path.join(ROOT, "include", "nasg.h")]
LIB = os.path.join(HERE, "libnasg_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-O2", "-I", os.path.join(ROOT, "include"), "-I", CSRC]


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or is_stale()):
        return LIB
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, os.path.basename(src).replace(".cu", ".o"))
        cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for cmd, pr in procs:
        out, _ = pr.communicate()
        if verbose or pr.returncode != 0:
            sys.stderr.write(out)
        if pr.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
