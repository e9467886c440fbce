"""In-tree build of the C-ABI CUDA library (sm_100a only): csrc/*.cu -> libxy_b200.so.

nvcc cross-compiles without a GPU, so this also runs on the CPU box (__graft_entry__.build()).
The .so is git-ignored but travels to the GPU box with the source snapshot.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libxy_b200.so")
SOURCES = ["xy_api.cu"]
HEADERS = ["xy_device.cuh", "xy_kernels.cuh", os.path.join("..", "..", "include", "xy.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
]


def _stale():
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force=False, verbose=False):
    if not force and not _stale():
        return LIB_PATH
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("XY_NVCC_EXTRA", "").split()          # e.g. -DXY_SWEEP_MIN_BLOCKS=3 when tuning
    cmd = [nvcc] + NVCC_FLAGS + extra + [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB_PATH]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libxy_b200.so (see output above)")
    with open(os.path.join(_HERE, "build_ptxas.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stderr)
    return LIB_PATH


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
