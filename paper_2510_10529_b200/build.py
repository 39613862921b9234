"""Build the C-ABI library in-tree: paper_2510_10529_b200/libfecheb.so (nvcc, sm_100a only, -lineinfo)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libfecheb.so")
SOURCES = ["fe_cheb.cu", "fe_tables.cpp", "fe_general.cpp"]
DEPS = SOURCES + ["fe_kernels.cuh", "fe_apply_tma.cuh", "fe_rr.cuh", "fe_minres.cuh", "fe_density.cuh", "fe_diag.cuh", "fe_general.cuh", "fe_gbox.cuh", "fe_general.h", "fe_tables.h", os.path.join("..", "..", "include", "fe_cheb.h")]


def nvcc_command(extra=()):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    return [nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
            "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", *extra,
            "-o", SO] + [os.path.join(CSRC, s) for s in SOURCES]


def build(force=False, verbose=False):
    newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in DEPS)
    if not force and os.path.exists(SO) and os.path.getmtime(SO) >= newest:
        return SO
    cmd = nvcc_command(("-Xptxas", "-v") if verbose else ())
    subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
