"""Builds libmg_b200.so (hand-written CUDA for sm_100a + host setup) in-tree with nvcc."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmg_b200.so")
SOURCES = ["mg_api.cu", "mg_kernels.cu", "mg_smoother.cu", "mg_coarse.cu", "mg_krylov.cu", "mg_tail.cu", "mg_bicgstab.cu", "mg_noalloc.cu", "mg_devinfo.cu", "mg_host_setup.cpp"]
HEADERS = ["mg_common.h", "mg_device.h", "mg_tile_gs.cuh", "mg_tile_ops.cuh", os.path.join("..", "..", "include", "mg_b200.h")]
NVCC_FLAGS = ["--threads", "0", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--shared", "-cudart", "shared"]


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + srcs
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
