"""Build libdgpe.so (the CUDA library behind include/dgpe.h) in-tree with nvcc for sm_100a.

Usage: python -m paper_1610_05329_b200.build [--force] [--verbose]
nvcc cross-compiles without a GPU; the built .so is git-ignored but travels with the tree.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdgpe.so")
SOURCES = ["dgpe_api.cu"]
DEPS = ["dgpe_api.cu", "common.cuh", "fft.cuh", "ctfft.cuh", "xyfft.cuh", "xysweep.cuh", "xysweep_tma.cuh", "xyfft_tma.cuh", "xyfft_pair.cuh", "tma.cuh", "zline.cuh", "spectral.cuh", "sweep.cuh", "observe.cuh"]
HEADER = os.path.join(os.path.dirname(HERE), "include", "dgpe.h")

# (no -split-compile: measured on the B200, the kernels it produces are slower -- x sweep 0.83 -> 0.96 ms,
# K3 0.67 -> 0.70 ms at 512^3 -- although it halves the build time)
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-shared", "-Xcompiler", "-fPIC",
    "-cudart", "static",
]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


STAMP = LIB + ".srchash"


def source_hash():
    """sha256 over the sources, the public header, this script and the flags: what libdgpe.so was built from.
    (Not modification times: a copied tree -- gpurun, a fresh checkout -- keeps contents, not mtimes.)"""
    import hashlib
    h = hashlib.sha256()
    for path in [os.path.join(CSRC, d) for d in sorted(DEPS)] + [HEADER, os.path.abspath(__file__)]:
        with open(path, "rb") as f:
            h.update(f.read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def up_to_date():
    if not (os.path.exists(LIB) and os.path.exists(STAMP)):
        return False
    with open(STAMP) as f:
        return f.read().strip() == source_hash()


def build(force=False, verbose=False):
    """Compile csrc/*.cu into paper_1610_05329_b200/libdgpe.so; returns its path."""
    if not force and up_to_date():
        return LIB
    cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libdgpe.so")
    with open(STAMP, "w") as f:
        f.write(source_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
