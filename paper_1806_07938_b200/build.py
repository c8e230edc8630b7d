"""Build libtomo_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1806_07938_b200.build [--force]

The shared library is the C-ABI boundary of include/tomo.h; the Python binding (tomo.py) loads it with ctypes.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtomo_b200.so")
OBJ = os.path.join(HERE, "build")

PERSIST_SIZES = [16, 20, 24, 32, 40, 64, 128, 160, 192, 256]     # TOMO_PERSIST_SIZES in csrc/persist_host.cuh
CU = [("tomo_api.cu", "tomo_api", []), ("solve_persistent.cu", "solve_persistent", []), ("lo_path.cu", "lo_path", [])] + \
     [("persist_inst.cu", f"persist_inst_{p}", [f"-DTOMO_PINST={p}"]) for p in PERSIST_SIZES]
CPP = ["host_model.cpp", "host_kernels.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-fopenmp", "-I", os.path.join(ROOT, "include"), "-I", CSRC]
CXX_FLAGS = ["-O2", "-std=c++17", "-fPIC", "-fopenmp", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
             "-I", "/usr/local/cuda/include"]


def _newest(paths):
    return max(os.path.getmtime(p) for p in paths)


def sources():
    out = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    out.append(os.path.join(ROOT, "include", "tomo.h"))
    out.append(os.path.join(ROOT, "include", "tomo_host.h"))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest(sources()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    objs = []
    procs = []
    jobs = []
    for f, stem, extra in CU:
        o = os.path.join(OBJ, stem + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *extra, "-c", os.path.join(CSRC, f), "-o", o]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        jobs.append(cmd)
        objs.append(o)
    for f in CPP:
        o = os.path.join(OBJ, f + ".o")
        jobs.append(["g++", *CXX_FLAGS, "-c", os.path.join(CSRC, f), "-o", o])
        objs.append(o)
    # at most one compiler per core at a time
    width = max(1, min(len(jobs), os.cpu_count() or 4))
    running = []
    pending = list(jobs)
    while pending or running:
        while pending and len(running) < width:
            cmd = pending.pop(0)
            running.append((cmd, subprocess.Popen(cmd)))
        cmd, p = running.pop(0)
        if p.wait() != 0:
            for _, q in running:
                q.kill()
            raise RuntimeError("build failed: " + " ".join(cmd))
    subprocess.check_call([nvcc, "-shared", "-o", LIB, *objs, "-Xcompiler", "-fopenmp", "-lgomp",
                           "-gencode", "arch=compute_100a,code=sm_100a"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
