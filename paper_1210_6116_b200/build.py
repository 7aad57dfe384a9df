"""Build paper_1210_6116_b200/libxy_b200.so: the C-ABI library of include/xy.h, sm_100a only.

nvcc cross-compiles without a GPU.  The library is built IN-TREE so that it travels with the
repository snapshot to the GPU box.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libxy_b200.so")
SOURCES = [os.path.join(CSRC, "xy_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "xy_kernels.cuh"), os.path.join(CSRC, "xy_device.cuh"),
                  os.path.join(CSRC, "potts_kernels.cuh"), os.path.join(CSRC, "potts_api.cuh"),
                  os.path.join(CSRC, "slab_kernels.cuh"),
                  os.path.join(HERE, "..", "include", "xy.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall", "-shared"]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("XY_NVCC_EXTRA", "").split()       # experiments only, e.g. -DKB_NW=12
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + SOURCES + ["-o", LIB]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
