"""Build the CUDA library (csrc/ -> libpca_b200.so, in-tree) for sm_100a with nvcc.

    python -m paper_0811_1081_b200.build [--force] [--verbose]

The .so is git-ignored but travels to the GPU box with the repo snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpca_b200.so")
SOURCES = [os.path.join(CSRC, "pca_api.cu"), os.path.join(CSRC, "pca_shard.cu"), os.path.join(CSRC, "pca_noalloc.cu")]
REG_INST = os.path.join(CSRC, "pca_reg_inst.cu")        # compiled REG_PARTS times with -DPCA_REG_PART=i
REG_PARTS = 6
HEADERS = [os.path.join(CSRC, f) for f in ("pca_device.cuh", "pca_solve.cuh", "pca_fused.cuh", "pca_tma.cuh", "pca_shard.cuh", "pca_reg.cuh", "pca_one.cuh",
                                           "pca_center.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "pca.h")]
OBJDIR = os.path.join(HERE, "build")


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    from concurrent.futures import ThreadPoolExecutor
    deps = SOURCES + HEADERS + [REG_INST]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    base = [nvcc_path(), "-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
            "-Xcompiler", "-fPIC"] + (["-Xptxas", "-v"] if verbose else [])
    jobs = [(src, os.path.join(OBJDIR, os.path.basename(src)[:-3] + ".o"), []) for src in SOURCES]
    jobs += [(REG_INST, os.path.join(OBJDIR, f"pca_reg_inst{i}.o"), [f"-DPCA_REG_PART={i}"]) for i in range(REG_PARTS)]

    def compile_one(job):
        src, obj, extra = job
        if force or not os.path.exists(obj) or any(os.path.getmtime(obj) < os.path.getmtime(d) for d in HEADERS + [src]):
            subprocess.run(base + extra + ["-c", src, "-o", obj], check=True)
        return obj

    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
        objs = list(ex.map(compile_one, jobs))
    subprocess.run([nvcc_path(), "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a",
                    "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
