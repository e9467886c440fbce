"""In-tree build of the C-ABI CUDA library (sm_100a only): csrc/*.cu -> libxy_b200.so.

nvcc cross-compiles without a GPU, so this also runs on the CPU box (__graft_entry__.build()).
The .so is git-ignored but travels to the GPU box with the source snapshot.  Staleness is decided by
a hash of every file under csrc/ and include/ plus the compiler flags, stored beside the library
(libxy_b200.so.hash): an edit to any kernel header rebuilds, a fresh checkout with new mtimes does not.
"""
import glob
import hashlib
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(_HERE, "..", "include")
LIB_PATH = os.path.join(_HERE, "libxy_b200.so")
HASH_PATH = LIB_PATH + ".hash"
SOURCES = ["xy_api.cu"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
]


def _extra_flags():
    return os.environ.get("XY_NVCC_EXTRA", "").split()          # e.g. -DXY_SWEEP_MIN_BLOCKS=3 when tuning


def dependencies():
    """Every file the library is compiled from: all of csrc/ and include/*.h."""
    deps = sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) +
                  glob.glob(os.path.join(INCLUDE, "*.h")))
    return [os.path.normpath(d) for d in deps]


def source_hash():
    h = hashlib.sha256()
    h.update(" ".join(NVCC_FLAGS + _extra_flags()).encode())
    for d in dependencies():
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def _stale():
    if not os.path.exists(LIB_PATH) or not os.path.exists(HASH_PATH):
        return True
    with open(HASH_PATH) as f:
        return f.read().strip() != source_hash()


def build_library(force=False, verbose=False):
    if not force and not _stale():
        return LIB_PATH
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + _extra_flags() + [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB_PATH]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libxy_b200.so (see output above)")
    with open(os.path.join(_HERE, "build_ptxas.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stderr)
    with open(HASH_PATH, "w") as f:
        f.write(source_hash() + "\n")
    return LIB_PATH


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
