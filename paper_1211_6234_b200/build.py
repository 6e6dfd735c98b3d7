"""Builds libdsmc.so (hand-written sm_100a CUDA behind the C ABI of include/dsmc.h) in-tree with nvcc."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdsmc.so")
SOURCES = ["dsmc_api.cu", "tensor_kernels.cu", "state_kernels.cu", "metropolis_kernels.cu", "sublattice_kernels.cu",
           "field_generic.cu", "field_tiled.cu", "field_fft.cu", "peak_kernels.cu", "wall_counts_noalloc.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--shared", "-cudart", "static", "--threads", "0"]


def _deps():
    d = [os.path.join(CSRC, s) for s in SOURCES]
    d.append(os.path.join(CSRC, "dsmc_internal.cuh"))
    d.append(os.path.join(CSRC, "bulk_copy.cuh"))
    d.append(os.path.join(CSRC, "packed_f32x2.cuh"))
    d.append(os.path.join(CSRC, "metropolis_common.cuh"))
    d.append(os.path.join(CSRC, "metropolis_pair.cuh"))
    d.append(os.path.join(HERE, "..", "include", "dsmc.h"))
    return d


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(p) for p in _deps()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
