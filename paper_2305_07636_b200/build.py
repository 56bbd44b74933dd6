"""Build the CUDA extension (sm_100a only) in-tree: csrc/libmcdc_b200.so."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libmcdc_b200.so")
SOURCES = ["mcdc_api.cu", "mcdc_transport.cu", "mcdc_comb.cu", "mcdc_pool.cu", "mcdc_noalloc.cu", "mcdc_device.cuh", "mcdc_kernels.cuh"]
# -fmad=false: no implicit contraction, every fma in the sources is explicit (DESIGN.md §3 C.2)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-fmad=false", "-lineinfo",
              "-std=c++17", "-Xcompiler", "-fPIC", "-shared"]


def stale():
    if not os.path.exists(LIB):
        return True
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [os.path.join(HERE, "..", "include", "mcdc.h")]
    return os.path.getmtime(LIB) < max(os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    if not force and not stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", LIB + ".tmp", os.path.join(CSRC, "mcdc_api.cu")]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
