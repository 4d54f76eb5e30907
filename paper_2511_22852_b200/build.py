"""Build libccake.so (hand-written CUDA for sm_100a) in-tree: paper_2511_22852_b200/libccake.so.

    python -m paper_2511_22852_b200.build [--force]

nvcc cross-compiles without a GPU.  -lineinfo keeps the source mapping for ncu's source page.  FMA contraction
stays on (default) for speed; the expressions that must be reproducible bit by bit (cell index, r^2 < (2h)^2)
use __dmul_rn / __dadd_rn explicitly (DESIGN.md §"Bit-exact decisions").
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libccake.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-O2", "--expt-relaxed-constexpr", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "ccake.h")]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(OUT) and os.path.getmtime(OUT) >= max(os.path.getmtime(p) for p in _deps()):
        return OUT
    extra = os.environ.get("CCAKE_NVCC_EXTRA", "").split()      # experiments only, e.g. -DCCAKE_PAIR_LPS=1
    cmd = [NVCC] + FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", OUT] + sources()
    subprocess.run(cmd, check=True)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
