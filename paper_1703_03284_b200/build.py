"""Build libmipwa.so (CUDA, sm_100a only) in-tree with nvcc.  `python -m paper_1703_03284_b200.build [--force]`.

The heavily specialised kernel families live in their own translation units (csrc/tu_*.cu, csrc/launch.h); the
objects are compiled in parallel and linked into one shared library."""
import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
UNITS = ["mipwa.cu", "tu_recompute.cu", "tu_recompute_mix.cu", "tu_abs2.cu", "tu_grad.cu", "tu_grad_mix.cu", "tu_grad_shp.cu",
         "tu_hybrid.cu"]
LIB = os.path.join(HERE, "libmipwa.so")
OBJ_DIR = os.path.join(HERE, "_obj")
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu*")) + glob.glob(os.path.join(CSRC, "*.h"))) + \
        [os.path.join(HERE, "..", "include", "mipwa.h")]


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in sources()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ_DIR, exist_ok=True)
    flags = NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else [])

    def compile_unit(u):
        obj = os.path.join(OBJ_DIR, u.replace(".cu", ".o"))
        subprocess.run([nvcc] + flags + ["-c", "-o", obj, os.path.join(CSRC, u)], check=True)
        return obj
    with ThreadPoolExecutor(max_workers=len(UNITS)) as pool:
        objs = list(pool.map(compile_unit, UNITS))
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
