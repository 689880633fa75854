"""Build the CUDA library (csrc/agnvar.cu -> libagnvar.so, in-tree) with nvcc for sm_100a.

Usage:  python -m paper_1909_06374_b200._build [--force]
nvcc cross-compiles without a GPU; the built .so travels to the GPU box with the repo snapshot.
"""
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libagnvar.so")
HASHFILE = LIB + ".hash"
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
]


def _sources():
    out = []
    for root, _, files in os.walk(CSRC):
        for f in files:
            if f.endswith((".cu", ".cuh", ".h")):
                out.append(os.path.join(root, f))
    out.append(os.path.join(INCLUDE, "agnvar.h"))
    return out


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def source_hash() -> str:
    """sha256 over the library's sources (names and contents): the staleness test of the built .so.  It is compiled
    into the library (agnvar_version() ends with it) and kept in a sidecar file next to the .so, so that neither a
    checkout nor a copy to another machine (which reset mtimes) can make a stale library look fresh."""
    h = hashlib.sha256()
    for path in sorted(_sources()):
        h.update(os.path.relpath(path, os.path.dirname(HERE)).encode())
        with open(path, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def is_fresh() -> bool:
    try:
        with open(HASHFILE) as f:
            return os.path.exists(LIB) and f.read().strip() == source_hash()
    except OSError:
        return False


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the sources changed since the .so was built.  Raises FileNotFoundError when nvcc is absent and
    subprocess.CalledProcessError when the compilation fails (a stale .so is never silently used for edited sources)."""
    if (not force) and is_fresh():
        return LIB
    digest = source_hash()
    cmd = [_nvcc()] + NVCC_FLAGS + [f'-DAGNVAR_SRC_HASH="{digest}"', "-I", INCLUDE, "-o", LIB,
                                    os.path.join(CSRC, "agnvar.cu")]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    subprocess.run(cmd, check=True)
    with open(HASHFILE, "w") as f:
        f.write(digest + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
