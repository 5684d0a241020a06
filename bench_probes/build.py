"""Builds bench_probes/libspiir_probe.so (sm_100a) — measurement helpers of bench.py only."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "probe.cu")
LIB = os.path.join(HERE, "libspiir_probe.so")


def build(force=False):
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    nvcc = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
                    "-Xcompiler", "-fPIC", "-o", LIB, SRC], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
