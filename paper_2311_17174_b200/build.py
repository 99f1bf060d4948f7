"""Compile the CUDA sources for sm_100a into shared libraries next to this file (in-tree, so they travel to the GPU box):
  csrc/emri.cu + csrc/loglike_static.cu -> libemri_b200.so   the product: the C ABI of include/emri.h
  csrc/probe.cu -> libemri_probe.so  bench.py's peak probes (include/emri_probe.h; not part of the boundary)
`python -m paper_2311_17174_b200.build [--force] [-v]`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
INC = os.path.join(os.path.dirname(HERE), "include")
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libemri_b200.so")
LIB_PROBE = os.path.join(HERE, "libemri_probe.so")
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-diag-suppress", "550"]
TARGETS = (
    (LIB, ("emri.cu", "loglike_static.cu"), ["-lcufft"],
     lambda: [os.path.join(INC, "emri.h")] + [os.path.join(CSRC, f) for f in os.listdir(CSRC)
                                              if f.endswith(".cuh") or f in ("emri.cu", "loglike_static.cu")]),
    (LIB_PROBE, ("probe.cu",), [], lambda: [os.path.join(INC, "emri_probe.h"), os.path.join(CSRC, "probe.cu")]),
)


def nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if c and os.path.exists(c):
            return c
    return "nvcc"


def _stale(lib, deps):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(f) > t for f in deps)


def stale():
    return any(_stale(lib, deps()) for lib, _, _, deps in TARGETS)


def build(force=False, verbose=False):
    for lib, src, libs, deps in TARGETS:
        if force or _stale(lib, deps()):
            cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [os.path.join(CSRC, f) for f in src] + ["-o", lib] + libs
            subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
