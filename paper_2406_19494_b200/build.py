"""Build libjf.so (the CUDA library behind include/jf.h) in-tree with nvcc for sm_100a."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libjf.so")
SOURCES = [os.path.join(HERE, "csrc", "jf_api.cu")]
DEPS = SOURCES + [os.path.join(HERE, "csrc", f) for f in ("jf_kernels.cuh", "jf_math.cuh", "jf_dual.cuh", "jf_tma.cuh", "jf_pc.cuh", "jf_f32x2.cuh")] + [
    os.path.join(ROOT, "include", "jf.h"), os.path.abspath(__file__)]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-cudart", "shared"]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in DEPS)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
    subprocess.check_call(cmd, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
