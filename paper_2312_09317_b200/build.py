"""Build step of the CUDA library (sm_100a only).  `python -m paper_2312_09317_b200.build`
or __graft_entry__.build().  nvcc cross-compiles without a GPU."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "csrc", "cpm_lib.cu")]
DEPS = SRC + [os.path.join(HERE, "csrc", "cpm_device.cuh"), os.path.join(HERE, "csrc", "cpm_pool_kernel.cuh"), os.path.join(HERE, "csrc", "cpm_stats_kernels.cuh"), os.path.join(os.path.dirname(HERE), "include", "cpm.h")]
LIB = os.path.join(HERE, "libcpm_b200.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def is_stale():
    return (not os.path.exists(LIB)) or any(os.path.getmtime(d) > os.path.getmtime(LIB) for d in DEPS)


def build(force=False, verbose=False):
    if not (force or is_stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = LIB + ".%d.tmp" % os.getpid()
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SRC
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
