"""Build libblink.so (the C-ABI library, include/blink.h) and libblink_testing.so (the same plus the test hooks of
include/blink_testing.h) for sm_100a, in-tree.

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
    if not (os.path.exists(LIB) and os.path.exists(os.path.join(HERE, "libblink_testing.so"))):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


# translation units that also hold test hooks (include/blink_testing.h) behind BLINK_TESTING_HOOKS: compiled a
# second time with the macro for libblink_testing.so -- the same library plus the host models and the fp32
# probe.  libblink.so itself is the product ABI (include/blink.h) only: no CPU model of any kernel is in it.
HOOK_SOURCES = ["blink_plan.cu", "blink_fused.cu", "blink_image_r.cu", "blink_probe.cu"]
TESTING_LIB = os.path.join(HERE, "libblink_testing.so")


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or _stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ_DIR, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []

    def compile_one(job):          # one translation unit -> object file (the units compile in parallel)
        src, hooks = job
        obj = os.path.join(OBJ_DIR, src.replace(".cu", ".hooks.o" if hooks else ".o"))
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-DBLINK_TESTING_HOOKS"] if hooks else []) + ["-c", os.path.join(CSRC, src), "-o", obj]
        return src, hooks, obj, subprocess.run(cmd, capture_output=True, text=True)

    jobs = [(s, False) for s in SOURCES if s != "blink_probe.cu"] + [(s, True) for s in HOOK_SOURCES]
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
        results = list(ex.map(compile_one, jobs))
    for *_, res in results:
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
    if any(res.returncode != 0 for *_, res in results):
        raise RuntimeError("nvcc failed building libblink.so")
    product = [obj for _, hooks, obj, _ in results if not hooks]
    testing = [obj for src, hooks, obj, _ in results if hooks] + \
              [obj for src, hooks, obj, _ in results if not hooks and src not in HOOK_SOURCES]
    for objs, lib in ((testing, TESTING_LIB), (product, LIB)):      # libblink.so last: _stale() looks at it
        link = subprocess.run([nvcc, "-shared", "-Xcompiler", "-pthread", "-gencode", "arch=compute_100a,code=sm_100a"] +
                              objs + ["-o", lib], capture_output=True, text=True)
        if link.returncode != 0:
            sys.stderr.write(link.stdout + link.stderr)
            raise RuntimeError(f"nvcc failed linking {os.path.basename(lib)}")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
