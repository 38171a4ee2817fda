"""Build liboptimus_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import glob
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(_HERE)
LIB = os.path.join(_HERE, "liboptimus_b200.so")
TRACE_LIB = os.path.join(_HERE, "liboptimus_b200_trace.so")   # -DOPTB_GEMM_TRACE: wait-cycle counters in the grouped GEMM (bench.py --side gemm_trace)
SRCS = sorted(glob.glob(os.path.join(_HERE, "csrc", "*.cu")))
HDRS = sorted(glob.glob(os.path.join(_HERE, "csrc", "*.h")) + glob.glob(os.path.join(_HERE, "csrc", "*.cuh"))) + [os.path.join(ROOT, "include", "optimus_b200.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def up_to_date(lib=LIB):
    if not os.path.exists(lib):
        return False
    t = os.path.getmtime(lib)
    return all(os.path.getmtime(f) <= t for f in SRCS + HDRS)


def build(force=False, verbose=False, trace=False):
    """trace=True builds the separate pipeline-trace library (never loaded by the product path)."""
    lib = TRACE_LIB if trace else LIB
    if not force and up_to_date(lib):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-DOPTB_GEMM_TRACE"] if trace else []) + (["-Xptxas", "-v"] if verbose else []) + \
          ["-I", os.path.join(ROOT, "include"), "-o", lib] + SRCS
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv))
