"""Build libblink.so (the C-ABI library, include/blink.h) for sm_100a, in-tree.

    python -m paper_2405_13478_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so lands next to this file so it travels with the repo
snapshot to the GPU box (it is git-ignored, not gpurun-ignored).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libblink.so")
SOURCES = ["blink_plan.cu", "blink_grid.cu", "blink_image.cu", "blink_image_w.cu", "blink_image_r.cu", "blink_fused.cu", "blink_fused_d4.cu", "blink_fused_tc.cu", "blink_correct.cu", "blink_dynspec.cu", "blink_probe.cu", "blink_host.cu"]
HEADERS = ["blink_internal.h", "parallel_for.h", "fft_core.cuh", "sphase.cuh", "sgather.cuh", "wfft.cuh", "fused_kernel.cuh", "fused_tc_kernel.cuh", os.path.join("..", "..", "include", "blink.h"),
           os.path.join("..", "..", "include", "blink_testing.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-pthread", "--expt-extended-lambda", "--expt-relaxed-constexpr"]
OBJ_DIR = os.path.join(HERE, "build")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or _stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ_DIR, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []

    def compile_one(src):          # one translation unit -> object file (the units compile in parallel)
        obj = os.path.join(OBJ_DIR, src.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + extra + ["-c", os.path.join(CSRC, src), "-o", obj]
        return obj, subprocess.run(cmd, capture_output=True, text=True)

    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    for _, res in results:
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
    if any(res.returncode != 0 for _, res in results):
        raise RuntimeError("nvcc failed building libblink.so")
    link = subprocess.run([nvcc, "-shared", "-Xcompiler", "-pthread", "-gencode", "arch=compute_100a,code=sm_100a"] +
                          [obj for obj, _ in results] + ["-o", LIB], capture_output=True, text=True)
    if link.returncode != 0:
        sys.stderr.write(link.stdout + link.stderr)
        raise RuntimeError("nvcc failed linking libblink.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
