"""Builds the C-ABI shared library `libs2w.so` in-tree with nvcc for sm_100a (no GPU needed to compile)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libs2w.so")
SOURCES = ["plan.cu", "wigner.cu", "ring_fft.cu", "fft16_kernels.cu", "pfa255_kernels.cu", "pfa4095_kernels.cu", "radial.cu", "filters.cpp"]
HEADERS = ["common.cuh", "fft_core.cuh", "fft16_core.cuh", "smem_attr.cuh", "pfa255_dft17.inc", "pfa4095_dft.inc", "pfa2047_dft.inc", "kernels.h", "host_math.h", os.path.join("..", "..", "include", "s2w.h")]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps if os.path.exists(d))


def build(force=False, verbose=False):
    """nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo ... -> libs2w.so (cudart linked statically)."""
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    for src in SOURCES:
        path = os.path.join(CSRC, src)
        if not os.path.exists(path):
            continue
        obj = os.path.join(CSRC, os.path.splitext(src)[0] + ".o")
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
               "-Xcompiler", "-fPIC,-O2", "-c", path, "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.check_call(cmd)
        objs.append(obj)
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static",
                           "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
