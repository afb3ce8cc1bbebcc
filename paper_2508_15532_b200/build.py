"""Build librt_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2508_15532_b200.build [--force] [--verbose]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librt_b200.so")
SOURCES = ["rt_api.cu", "rt_transport.cu", "rt_transport_tile.cu", "rt_source.cu", "rt_moments_mma.cu", "rt_angular_mapr.cu", "rt_geodesic.cpp", "rt_geometry.cpp"]
HEADERS = ["rt_internal.h", "rt_kernels.cuh", "rt_transport_dev.cuh", os.path.join("..", "..", "include", "rt.h")]


def stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force=False, verbose=False):
    if not (force or stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
           "-Xcompiler", "-fPIC", "--fmad=true", "-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
