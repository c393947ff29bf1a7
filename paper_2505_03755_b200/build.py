"""Build libdfjk.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2505_03755_b200.build [--force]

Every .cu is compiled to an object file in parallel, then linked into one shared library.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
SOURCES = ["api.cu", "prep.cu", "jpass.cu", "kpath.cu", "ao2mo.cu", "emu.cu", "symm.cu", "small.cu"]
HEADERS = ["common.cuh", "ctx.h", "pipeline.cuh", os.path.join("..", "..", "include", "dfjk.h")]
LIB = os.path.join(HERE, "libdfjk.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)

    def compile_one(src: str):
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + ["-c", "-o", obj, os.path.join(CSRC, src)]
        return obj, subprocess.run(cmd, capture_output=True, text=True)

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    log = "".join(r.stdout + r.stderr for _, r in results)
    failed = [r for _, r in results if r.returncode != 0]
    if verbose or failed:
        sys.stderr.write(log)
    if failed:
        raise RuntimeError("nvcc failed building libdfjk.so")
    link = subprocess.run([nvcc, "-shared", "-o", LIB] + [o for o, _ in results], capture_output=True, text=True)
    if link.returncode != 0:
        sys.stderr.write(link.stdout + link.stderr)
        raise RuntimeError("nvcc failed linking libdfjk.so")
    with open(os.path.join(HERE, "ptxas_info.log"), "w") as f:
        f.write(log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
