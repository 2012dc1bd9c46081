"""Build the CUDA C-ABI library in-tree: paper_1104_3998_b200/libpic1d.so (sm_100a only).

-fmad=false: every fp32 operation is the IEEE operation that is written (explicit __fmaf_rn where
the step definition says fma), so discrete outputs (keys, offsets, masks) match the oracle bit for
bit.  No fast-math; IEEE division and square root (nvcc defaults).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpic1d.so")
SOURCES = ["pic1d.cu", "pic1d_gsort.cu", "pic1d_field_static.cu"]
DEPS = sorted(f for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh")))   # every source under csrc/
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-fmad=false",
              "-std=c++17", "-shared", "-Xcompiler", "-fPIC"]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, d) for d in DEPS] + [os.path.join(HERE, "..", "include", h) for h in ("pic1d.h", "pic1d_gsort.h", "pic1d_static.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + \
        [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
