"""Build the product library (CUDA kernels + C-ABI) for sm_100a, in-tree.

    python -m paper_1501_03869_b200.build        ->  paper_1501_03869_b200/libpat_b200.so

nvcc cross-compiles without a GPU.  -fmad=false is NOT used: contraction-sensitive
expressions in the kernels are written with explicit __f*_rn intrinsics instead.
"""
import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpat_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-shared", "-Xcompiler", "-fPIC,-fopenmp,-O3,-Wall", "-cudart", "static", "--threads", "0"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cpp")))


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> str:
    srcs = sources()
    deps = srcs + glob.glob(os.path.join(CSRC, "*.h")) + [os.path.join(HERE, "..", "include", "pat.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    extra = os.environ.get("PAT_NVCC_FLAGS", "").split()          # experiments: e.g. PAT_NVCC_FLAGS=-DPAT_LEGACY_LAYOUTS=1
    cmd = [NVCC, *FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), *(["-DPAT_TRACE_BUILD"] if trace else []),
           "-o", tmp, *srcs, "-lgomp"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv, trace="--trace" in sys.argv))   # --trace: PAT_TRACE_FILE timeline
