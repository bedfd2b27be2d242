"""Build paper_1910_12578_b200/libcst.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

Usage: python -m paper_1910_12578_b200.build [--force]
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcst.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
         "-Xcompiler", "-fPIC", "--shared"]
# The operators beyond the graded path whose Riemann problems at a reflecting wall must see EXACT mirror images (the
# upwind side is decided on a sum that cancels exactly there: DESIGN.md reading Q6b) are compiled without FMA
# contraction: a product fused into one of two mirror-image formulas and not into the other breaks the cancellation.
# They are multi-pass, untuned kernels; the hot kernels keep nvcc's default.
PER_FILE = {"ctu.cu": ["-fmad=false"], "fourth.cu": ["-fmad=false"]}


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(HERE, "..", "include", "*.h"))
    return any(os.path.getmtime(f) > t for f in deps)


def build(force=False, verbose=False):
    """Compile every csrc/*.cu to an object file (in parallel) and link libcst.so."""
    if not force and not needs_build():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    cflags = [f for f in FLAGS if f != "--shared"] + (["-Xptxas", "-v"] if verbose else []) + \
        os.environ.get("CST_NVCC_EXTRA", "").split()

    def compile_one(src):
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        subprocess.run([NVCC] + cflags + PER_FILE.get(os.path.basename(src), []) + ["-c", "-o", obj, src], check=True)
        return obj
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        objs = list(ex.map(compile_one, sources()))
    subprocess.run([NVCC, "--shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
