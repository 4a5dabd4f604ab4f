"""Builds libgeoclaw_b200.so (the CUDA path) in-tree with nvcc for sm_100a.

    python -m paper_1901_06798_b200.build

-fmad=false: no FMA contraction beyond the explicit __fma_rn calls DESIGN.md section 3 specifies, so the kernels
evaluate it bit-for-bit (IEEE divide and sqrt are nvcc's defaults for fp64).  -lineinfo keeps the ncu source page usable.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = ["gc_api.cu", "gc_api_amr.cu", "gc_sweep.cu", "gc_ghost.cu", "gc_amr.cu", "gc_unsplit.cu"]
LIB = os.path.join(HERE, "libgeoclaw_b200.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-fmad=false", "-std=c++17",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-O2", "-shared"]


def build(force=False, verbose=False):
    srcs = [os.path.join(HERE, "csrc", s) for s in SRC if os.path.exists(os.path.join(HERE, "csrc", s))]
    inc = os.path.join(HERE, "..", "include")
    deps = srcs + [os.path.join(HERE, "csrc", h) for h in sorted(os.listdir(os.path.join(HERE, "csrc"))) if h.endswith((".h", ".cuh"))] + \
        [os.path.join(inc, h) for h in sorted(os.listdir(inc)) if h.endswith(".h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + srcs
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
