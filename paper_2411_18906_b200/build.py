"""Builds libhea_b200.so in-tree with nvcc for sm_100a (the only target).  `python -m paper_2411_18906_b200.build`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhea_b200.so")
SOURCES = ["hea_api.cu", "hea_sro.cu", "hea_mc.cu", "hea_mc2.cu", "hea_mc2_p1.cu", "hea_mc2_p2.cu", "hea_mc2_p3.cu", "hea_pool.cu", "hea_lattice.cpp"]
HEADERS = ["hea_mc2.cu", "hea_device.cuh", "hea_mc_common.cuh", "hea_lattice.hpp", os.path.join("..", "..", "include", "hea.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-pthread", "-shared", "--threads", "0"]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile every CUDA source of the package for sm_100a into one shared library.  Returns its path."""
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []),
           *[os.path.join(CSRC, s) for s in SOURCES], "-o", LIB]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
