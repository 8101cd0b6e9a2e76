"""Build libmipwa.so (CUDA, sm_100a only) in-tree with nvcc.  `python -m paper_1703_03284_b200.build [--force]`."""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "mipwa.cu")
LIB = os.path.join(HERE, "libmipwa.so")
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-shared",
              "-Xcompiler", "-fPIC"]


def sources():
    return sorted(f for f in glob.glob(os.path.join(HERE, "csrc", "*.cu*")) if not f.endswith("fp64_microbench.cu")) \
        + [os.path.join(HERE, "..", "include", "mipwa.h")]


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in sources()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


def build_microbench():
    """Stand-alone FP64-pipe microbenchmarks (csrc/fp64_microbench.cu -> ./fp64_microbench); not part of the library."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    out = os.path.join(HERE, "fp64_microbench")
    subprocess.run([nvcc, "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-o", out,
                    os.path.join(HERE, "csrc", "fp64_microbench.cu")], check=True)
    return out


if __name__ == "__main__":
    if "--microbench" in sys.argv:
        print(build_microbench())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
