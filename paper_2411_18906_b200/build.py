"""Builds libhea_b200.so in-tree with nvcc for sm_100a (the only target).  `python -m paper_2411_18906_b200.build`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhea_b200.so")
SOURCES = ["hea_api.cu", "hea_sro.cu", "hea_sro2.cu", "hea_mc.cu", "hea_mc2.cu", "hea_mc2_p1.cu", "hea_mc2_p2.cu", "hea_mc2_p3.cu", "hea_pool.cu", "hea_peaks.cu", "hea_noalloc.cu", "hea_lattice.cpp"]
HEADERS = ["hea_mc2.cu", "hea_device.cuh", "hea_mc_common.cuh", "hea_lattice.hpp", os.path.join("..", "..", "include", "hea.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-pthread"]
OBJDIR = os.path.join(HERE, "build")            # per-source objects (git-ignored), so an edit recompiles one file


def _newer(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _stale():
    return _newer(LIB, [os.path.join(CSRC, s) for s in SOURCES + HEADERS])


def build(force=False, verbose=False):
    """Compile every CUDA source of the package for sm_100a (one object per source, in parallel) and link them into
    one shared library.  Returns its path."""
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJDIR, exist_ok=True)
    headers = [os.path.join(CSRC, h) for h in HEADERS]
    jobs, objs = [], []
    for src in SOURCES:
        obj = os.path.join(OBJDIR, os.path.splitext(src)[0] + ".o")
        objs.append(obj)
        if force or _newer(obj, [os.path.join(CSRC, src), *headers]):
            cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c", os.path.join(CSRC, src), "-o", obj]
            jobs.append((cmd, subprocess.Popen(cmd)))
    for cmd, proc in jobs:
        if proc.wait() != 0:
            raise subprocess.CalledProcessError(proc.returncode, cmd)
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-pthread",
                           *objs, "-o", LIB])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
