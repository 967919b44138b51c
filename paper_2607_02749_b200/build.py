"""In-tree build of libgvqe.so (nvcc, sm_100a only).  ``python -m paper_2607_02749_b200.build`` or build().

Every source is compiled to an object under build/ (in parallel, only when it or a header is newer), then linked."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
SO = os.path.join(HERE, "libgvqe.so")
SOURCES = ["schedule.cpp", "lower.cpp", "hamiltonian.cpp", "graph.cpp", "cobyla.cpp", "driver.cpp", "jit.cpp", "jit_expect.cpp", "jit_rt.cpp", "gvqe_api.cpp",
           "kernels.cu", "expect.cu"]
HEADERS = ["program.h", "devprog.h", "schedule.h", "lower.h", "hamiltonian.h", "graph.h", "cobyla.h", "kernels.h", "kernels.cuh", "jit.h", "jit_internal.h",
           os.path.join("..", "..", "include", "gvqe.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CFLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]
LFLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-cudart", "static", "-ldl", "-lpthread"]


def _sources():
    return [s for s in SOURCES if os.path.exists(os.path.join(CSRC, s))]


def _newest_header() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS if os.path.exists(os.path.join(CSRC, h)))


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in _sources()) or _newest_header() > t


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return SO
    os.makedirs(OBJ, exist_ok=True)
    th = _newest_header()
    jobs = []
    for s in _sources():
        src, obj = os.path.join(CSRC, s), os.path.join(OBJ, s + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), th):
            jobs.append([NVCC] + CFLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src])
    with ThreadPoolExecutor(max_workers=8) as ex:
        for rc in ex.map(lambda c: subprocess.call(c), jobs):
            if rc:
                raise RuntimeError("nvcc failed")
    tmp = SO + f".tmp{os.getpid()}"
    subprocess.check_call([NVCC] + LFLAGS + ["-o", tmp] + [os.path.join(OBJ, s + ".o") for s in _sources()])
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
