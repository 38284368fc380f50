"""Build step of the CUDA path: nvcc -> libising_b200.so, in-tree, sm_100a only.

Used by __graft_entry__.build() and, when the library is missing or stale, by binding.py.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libising_b200.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC",
              "-diag-suppress", "128"]   # "loop is not reachable": the evaluation instantiation of row_update returns early


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))
                  + glob.glob(os.path.join(os.path.dirname(_HERE), "include", "*.h")))


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def nvcc_path():
    return shutil.which("nvcc") or ("/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else None)


def build_library(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu under csrc/ into libising_b200.so (one translation unit: ising_api.cu)."""
    if not force and not is_stale():
        return LIB
    nvcc = nvcc_path()
    if nvcc is None:
        raise RuntimeError("nvcc not found: cannot build libising_b200.so (there is no CPU fallback)")
    tuning = ["-DISING_TUNING_ENV"] if os.environ.get("ISING_BUILD_TUNING") == "1" else []   # env knobs: tuning builds only
    cmd = [nvcc] + NVCC_FLAGS + tuning + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", LIB + ".tmp", os.path.join(CSRC, "ising_api.cu")]
    subprocess.check_call(cmd)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
