"""Builds libomnimem.so (the C-ABI library of include/omnimem.h) in-tree with nvcc for sm_100a.

    python -m paper_2605_30519_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so stays next to this file (git-ignored, but it travels
with the tree), so nothing depends on a JIT cache.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libomnimem.so")
SOURCES = ["omnimem_api.cu", "cache_kernels.cu", "select_kernels.cu", "attn_tcgen05.cu", "offload.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr",
         *os.environ.get("OMNIMEM_NVCC_FLAGS", "").split()]


def _deps_mtime() -> float:
    m = os.path.getmtime(os.path.join(HERE, "..", "include", "omnimem.h"))
    for f in os.listdir(CSRC):
        m = max(m, os.path.getmtime(os.path.join(CSRC, f)))
    return m


def build(force: bool = False, verbose: bool = False, out: str | None = None, extra_flags=()) -> str:
    """``out`` / ``extra_flags``: build a variant (e.g. ``-DOMNIMEM_TRACE``) beside the product library; a process
    picks it up through the ``OMNIMEM_LIB`` environment variable (binding.py)."""
    LIB = out or globals()["LIB"]
    OBJ = globals()["OBJ"] if out is None else out + ".obj"
    FLAGS = [*globals()["FLAGS"], *extra_flags]
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _deps_mtime():
        return LIB
    os.makedirs(OBJ, exist_ok=True)

    def compile_one(src: str) -> str:
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        r = subprocess.run([NVCC, *FLAGS, "-c", os.path.join(CSRC, src), "-o", obj], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
        with open(obj + ".log", "w") as f:
            f.write(r.stdout + r.stderr)
        if verbose:
            print(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call([NVCC, "-shared", "-o", tmp, *objs, "-cudart", "static"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
