"""Builds libpwham.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.  No GPU is needed to build."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpwham.so")
SOURCES = ["pwham.cu", "local_kernels.cu", "local_fast.cu", "local_v2.cu", "local_z.cu", "zgemm.cu", "rr.cu", "rr_api.cu", "paw.cu", "lobpcg.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-O2", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "pwham.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    """One `nvcc -c` per translation unit (in parallel), then one link step.  Objects go to build/ (git-ignored)."""
    if not force and not needs_build():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    cflags = [f for f in NVCC_FLAGS if f != "-shared"] + (["-Xptxas", "-v"] if verbose else [])

    def compile_one(src: str):
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        res = subprocess.run([_nvcc()] + cflags + ["-c", "-o", obj, os.path.join(CSRC, src)], capture_output=True, text=True)
        return src, obj, res

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    for src, _, res in results:
        if verbose or res.returncode != 0:
            sys.stderr.write(f"--- {src}\n" + res.stdout + res.stderr)
    if any(res.returncode != 0 for _, _, res in results):
        raise RuntimeError("nvcc failed building libpwham.so")
    link = subprocess.run([_nvcc(), "-shared", "-o", LIB] + [obj for _, obj, _ in results], capture_output=True, text=True)
    if link.returncode != 0:
        sys.stderr.write(link.stdout + link.stderr)
        raise RuntimeError("nvcc failed linking libpwham.so")
    return LIB


if __name__ == "__main__":
    print(build_lib(force=True, verbose="-v" in sys.argv))
