"""Builds paper_2606_17065_b200/libpivot_iv.so (hand-written CUDA, sm_100a only) in-tree with nvcc.

nvcc cross-compiles without a GPU; the built .so travels to the GPU box with the repo snapshot.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SO = os.path.join(HERE, "libpivot_iv.so")
SRC = [os.path.join(HERE, "csrc", f) for f in ("pivot_iv.cu", "pivot_greeks.cu", "pivot_debug.cu")]
DEPS = SRC + [os.path.join(HERE, "csrc", "lbr_device.cuh"), os.path.join(HERE, "csrc", "coeffs.cuh"), os.path.join(ROOT, "include", "pivot_iv.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
         "-shared", "-cudart", "shared"]


SO_CHECKED = os.path.join(HERE, "libpivot_iv_boundscheck.so")


def needs_build(so: str = SO) -> bool:
    return not os.path.exists(so) or any(os.path.getmtime(so) < os.path.getmtime(d) for d in DEPS)


def build(force: bool = False, verbose: bool = False, bounds_check: bool = False) -> str:
    """bounds_check=True builds libpivot_iv_boundscheck.so: the same sources with -DPIVOT_BOUNDS_CHECK (device-side asserts on
    every shared-memory index of the tile kernel), loaded only by tests/test_gpu_boundscheck.py."""
    so = SO_CHECKED if bounds_check else SO
    if not force and not needs_build(so):
        return so
    cmd = [NVCC] + FLAGS + (["-DPIVOT_BOUNDS_CHECK"] if bounds_check else []) + (["-Xptxas", "-v"] if verbose else []) + ["-o", so] + SRC
    subprocess.check_call(cmd)
    return so


if __name__ == "__main__":
    print(build(force=True, verbose=True))
