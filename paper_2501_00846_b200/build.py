"""Build step for the CUDA library (nvcc, sm_100a only).  Used by __graft_entry__.build()."""
import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libtslb.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-cudart", "shared", "-shared", "-Xcompiler", "-fPIC",
              "-Xlinker", "-rpath=/usr/local/cuda/lib64", "-diag-suppress", "128"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))
                  + glob.glob(os.path.join(INCLUDE, "*.h")))


def stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def build_cuda(force=False, verbose=False):
    """Compile csrc/tslb_api.cu (which includes the kernel headers) into libtslb.so in-tree."""
    if not force and not stale():
        return LIB
    cmd = ["nvcc"] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [
        "-o", LIB, os.path.join(CSRC, "tslb_api.cu")]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    import sys
    build_cuda(force=True, verbose="-v" in sys.argv)
    print(LIB)
