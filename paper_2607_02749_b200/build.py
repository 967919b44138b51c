"""In-tree build of libgvqe.so (nvcc, sm_100a only).  ``python -m paper_2607_02749_b200.build`` or build()."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libgvqe.so")
SOURCES = ["schedule.cpp", "lower.cpp", "hamiltonian.cpp", "graph.cpp", "driver.cpp", "gvqe_api.cpp", "kernels.cu"]
HEADERS = ["program.h", "devprog.h", "schedule.h", "lower.h", "hamiltonian.h", "graph.h", "kernels.h", "kernels.cuh",
           os.path.join("..", "..", "include", "gvqe.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
         "-Xcompiler", "-fPIC", "-cudart", "static"]


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return SO
    tmp = SO + f".tmp{os.getpid()}"
    cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
