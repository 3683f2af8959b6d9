"""Compile and run the instruction-throughput microbenchmark csrc/fp32_peak.cu (needs a GPU to run).

Usage: python -m paper_2104_00537_b200.fp32_peak [--build-only]
It backs the FP32 roofline denominator of bench.py (148 SM x 128 lanes x 2 flop x SM clock) with a measured
FFMA issue rate; the table is kept under profiles/.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "fp32_peak.cu")
OUT = os.path.join(HERE, "csrc", "build", "fp32_peak")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build() -> str:
    os.makedirs(os.path.dirname(OUT), exist_ok=True)
    if not os.path.exists(OUT) or os.path.getmtime(OUT) < os.path.getmtime(SRC):
        subprocess.check_call([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
                               SRC, "-o", OUT])
    return OUT


if __name__ == "__main__":
    exe = build()
    if "--build-only" not in sys.argv:
        sys.exit(subprocess.call([exe]))
