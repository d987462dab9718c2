"""Build step: compiles csrc/ into libewald_b200.so next to this file (nvcc, sm_100a only).

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the tree to the GPU box.
Run as `python -m paper_2507_02888_b200.build [--force] [--verbose]`.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libewald_b200.so")
SOURCES = ["ewald_api.cu", "jastrow_api.cu", "blip_api.cu", "ewald_setup.cpp", "ewald_octplan.cpp"]
HEADERS = [os.path.join(ROOT, "include", "ewald.h"), os.path.join(ROOT, "include", "jastrow.h"), os.path.join(ROOT, "include", "blip.h"),
           os.path.join(CSRC, "ewald_internal.h"), os.path.join(CSRC, "jastrow_kernels.cuh"),
           os.path.join(CSRC, "ewald_recip_mma.cuh"),
           os.path.join(CSRC, "ewald_kernels.cuh"),
           os.path.join(CSRC, "ewald_kernels_common.cuh"), os.path.join(CSRC, "ewald_realspace.cuh"),
           os.path.join(CSRC, "ewald_recip_oct.cuh")]

# --split-compile is pinned: with =0 (one piece per host core) the register allocation of the big kernels, and with
# it 4-13 % of their speed, depended on the core count of the machine that built the library
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "--split-compile=1"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def stale():
    if not os.path.exists(LIB):
        return True
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return os.path.getmtime(LIB) < max(os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    """Compile the library if it is missing or older than its sources; returns its path."""
    if not (force or stale()):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-I", os.path.join(ROOT, "include"), "-I", CSRC, "-o", tmp] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    try:
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    finally:
        if os.path.exists(tmp):
            os.remove(tmp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
