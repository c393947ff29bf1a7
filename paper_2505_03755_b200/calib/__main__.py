"""Build and run the calibration microbenchmarks on cuda:0; prints their tables to stdout.

    python -m paper_2505_03755_b200.calib [peaks] [matmul]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
PROGRAMS = ["peaks"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17"]


def build(name: str) -> str:
    out = os.path.join(HERE, "build", name)
    os.makedirs(os.path.dirname(out), exist_ok=True)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc] + NVCC_FLAGS + ["-o", out, os.path.join(HERE, name + ".cu")], check=True)
    return out


def matmul_fp64() -> None:
    """cuBLAS fp64 GEMM through torch.matmul, 8192^3: burst (best of 10) and sustained (4 s). Calibration only."""
    import time
    import torch
    n = 8192
    a = torch.randn((n, n), dtype=torch.float64, device="cuda")
    b = torch.randn((n, n), dtype=torch.float64, device="cuda")
    for _ in range(2):
        a @ b
    best = 1e9
    for _ in range(10):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); a @ b; e1.record(); torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    t0, reps = time.perf_counter(), 0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    while time.perf_counter() - t0 < 4.0:
        a @ b
        reps += 1
        if reps % 8 == 0:
            torch.cuda.synchronize()
    e1.record(); torch.cuda.synchronize()
    print(f"cuBLAS fp64 matmul {n}^3: burst {2 * n ** 3 / best * 1e-9:.2f} TFLOP/s, "
          f"sustained {2 * n ** 3 * reps / e0.elapsed_time(e1) * 1e-9:.2f} TFLOP/s over {reps} calls")


def main(argv):
    todo = argv or PROGRAMS + ["matmul"]
    for name in todo:
        print(f"==== {name}", flush=True)
        if name == "matmul":
            matmul_fp64()
        else:
            subprocess.run([build(name)], check=True)
        sys.stdout.flush()


if __name__ == "__main__":
    main(sys.argv[1:])
