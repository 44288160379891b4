"""Build the CPU oracle (test infrastructure) into oracle/liboracle.so with gcc.

Usage: python oracle/build.py     (also called by __graft_entry__.build() and tests/conftest.py)
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dgpe_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")


STAMP = LIB + ".srchash"
CMD = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]


def source_hash() -> str:
    """sha256 of the oracle's sources and flags (contents, not modification times: copied trees keep only those)."""
    import hashlib
    h = hashlib.sha256()
    for path in (SRC, os.path.join(HERE, "dgpe_oracle.h")):
        with open(path, "rb") as f:
            h.update(f.read())
    h.update(" ".join(CMD[:-4]).encode())
    return h.hexdigest()


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.exists(STAMP):
        with open(STAMP) as f:
            if f.read().strip() == source_hash():
                return LIB
    subprocess.run(CMD, check=True)
    with open(STAMP, "w") as f:
        f.write(source_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
