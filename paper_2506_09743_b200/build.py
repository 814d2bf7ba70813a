"""Build libqmcb200.so in-tree with nvcc for sm_100a (no JIT cache: the built library
travels with the repository snapshot to the GPU box).  The template kernels are instantiated in one translation
unit per (NS, NMO) variant (csrc/qmc_variant_*.cu); the units are compiled in parallel and linked."""
from __future__ import annotations

import os
import shutil
import subprocess
import tempfile
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libqmcb200.so")
SOURCES = ["qmc_api.cu", "qmc_variant_7_14.cu", "qmc_variant_8_16.cu", "qmc_variant_4_8.cu", "qmc_variant_3_8.cu",
           "qmc_variant_2_2.cu", "qmc_variant_1_2.cu"]
HEADERS = ["qmc_device.cuh", "qmc_eval.cuh", "qmc_kernels.cuh", "qmc_backflow.cuh", "qmc_variant.cuh"]
INCLUDE = os.path.join(os.path.dirname(HERE), "include", "qmc.h")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [INCLUDE]
    return any(os.path.getmtime(f) > t for f in deps)


def build(force: bool = False, verbose: bool = False, extra_flags: list[str] | None = None, out: str | None = None) -> str:
    out = out or SO
    if out == SO and not (force or needs_build()):
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = FLAGS + (["-Xptxas=-v"] if verbose else []) + list(extra_flags or [])
    tmp = tempfile.mkdtemp(prefix="qmcb200_build_")
    try:
        def compile_one(src):
            obj = os.path.join(tmp, os.path.splitext(src)[0] + ".o")
            subprocess.check_call([nvcc] + flags + ["-c", os.path.join(CSRC, src), "-o", obj])
            return obj

        with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as ex:
            objs = list(ex.map(compile_one, SOURCES))
        subprocess.check_call([nvcc] + FLAGS[:2] + ["-shared", "-o", out] + objs)
    finally:
        shutil.rmtree(tmp, ignore_errors=True)
    return out


if __name__ == "__main__":
    print(build(force=True, verbose=True))
