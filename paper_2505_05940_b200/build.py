"""Build libmodal.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmodal.so")
SOURCES = [os.path.join(CSRC, "modal_api.cu"), os.path.join(CSRC, "vk_static.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("kernels.cuh", "host_math.hpp", "vk_flow.cuh", "flow_schedule.hpp", "vk_mma.cuh", "mma_schedule.hpp", "peaks.cuh", "vk_stream.cuh", "stream_schedule.hpp", "vk_bptt.cuh", "vk_small.cuh", "vk_dense.cuh", "vk_repl.cuh", "repl_schedule.hpp")] + [
    os.path.join(os.path.dirname(HERE), "include", "modal.h")]


def nvcc_cmd(out: str, extra=()):
    return ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
            "-shared", "-Xcompiler", "-fPIC",
            "--expt-relaxed-constexpr", *os.environ.get("MODAL_NVCC_FLAGS", "").split(), *extra, "-o", out, *SOURCES]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = nvcc_cmd(tmp, ("-Xptxas", "-v") if verbose else ())
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
