"""Builds libqft.so (the C-ABI library of include/qft.h) in-tree with nvcc for sm_100a.

    python -m paper_2606_18981_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libqft.so")
SOURCES = ["qft_api.cu", "qft_kernels.cu", "qft_tma_lt7.cu", "qft_tma_lt8.cu", "qft_tma_lt9.cu", "qft_tma_xt.cu", "qft_tma_es.cu", "qft_metrics.cu", "qft_metrics_static.cu", "qft_plan.cpp"]
HEADERS = ["qft_plan.h", "qft_device.cuh", "qft_fused.cuh", "qft_tma.cuh", "qft_tma_inst.cuh", "qft_packed.cuh", "qft_phase.cuh", "qft_launch.h", os.path.join("..", "..", "include", "qft.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "static",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    for f in SOURCES + HEADERS + [os.path.join("..", "build.py")]:
        p = os.path.join(CSRC, f)
        if os.path.exists(p) and os.path.getmtime(p) > t:
            return True
    return False


def build(force: bool = False, verbose: bool = False, extra_flags=(), lib: str = LIB) -> str:
    """Compile every source to an object file in parallel (one nvcc process each), then link.
    extra_flags / lib: a differently configured build beside the product's (e.g. -DQFT_PHASE_TIMING)."""
    if force or _stale() or lib != LIB:
        from concurrent.futures import ThreadPoolExecutor

        nvcc = os.environ.get("NVCC", "nvcc")
        objdir = os.path.join(HERE, "build" if lib == LIB else "build_" + os.path.basename(lib))
        os.makedirs(objdir, exist_ok=True)
        cflags = [f for f in NVCC_FLAGS if f not in ("-shared",)] + list(extra_flags)

        def compile_one(src: str) -> str:
            obj = os.path.join(objdir, os.path.splitext(src)[0] + ".o")
            cmd = [nvcc] + cflags + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
            subprocess.run(cmd, check=True)
            return obj

        with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
            objs = list(ex.map(compile_one, SOURCES))
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static",
                        "-o", lib] + objs, check=True)
    return lib


if __name__ == "__main__":
    # python -m paper_2606_18981_b200.build [--force] [-v] [--define NAME ... --lib PATH]: the product library, or a
    # differently configured one beside it (e.g. --define QFT_PHASE_TIMING --lib /tmp/libqft_phase.so for tune --phase-lib)
    defs = [sys.argv[i + 1] for i, a in enumerate(sys.argv[:-1]) if a == "--define"]
    alt = [sys.argv[i + 1] for i, a in enumerate(sys.argv[:-1]) if a == "--lib"]
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, extra_flags=["-D" + d for d in defs],
                lib=os.path.abspath(alt[0]) if alt else LIB))
