"""Build step of the CUDA library: nvcc -> paper_2504_04465_b200/liblbm_b200.so (in-tree, sm_100a only).

    python -m paper_2504_04465_b200.build [--force]

One object per translation unit (one per lattice, so the template instantiations compile in
parallel), then one shared library with the CUDA runtime linked statically, so that the library
loads (and the host grid builder runs) on machines without a GPU.
"""
import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liblbm_b200.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

CU = ["lbm_api.cu", "peak.cu", "sweep_q9.cu", "sweep_q13.cu", "sweep_q21.cu", "sweep_q37.cu"]
CPP = ["grid_builder.cpp"]
HEADERS = sorted(os.path.join(CSRC, h) for h in os.listdir(CSRC) if h.endswith((".cuh", ".hpp", ".h"))) + [os.path.join(INCLUDE, "lbm.h")]

NVCC = os.environ.get("NVCC", "nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ARCH + ["-std=c++17", "-O3", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]
CXX_FLAGS = ["-std=c++17", "-O2", "-fPIC", "-pthread"]


def _stale(target, deps):
    return not os.path.exists(target) or any(os.path.getmtime(d) > os.path.getmtime(target) for d in deps)


def _compile(src):
    obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
    path = os.path.join(CSRC, src)
    if src.endswith(".cu"):
        cmd = [NVCC] + NVCC_FLAGS + ["-c", path, "-o", obj]
    else:
        cmd = ["g++"] + CXX_FLAGS + ["-c", path, "-o", obj]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    with open(obj + ".log", "w") as fh:          # ptxas -v: registers / spills per kernel
        fh.write(" ".join(cmd) + "\n" + r.stdout)
    if r.returncode != 0:
        raise RuntimeError("compile failed: %s\n%s" % (" ".join(cmd), r.stdout[-4000:]))
    return obj


def build(force=False, verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    srcs = CU + CPP
    objs = [os.path.join(OBJ, os.path.splitext(s)[0] + ".o") for s in srcs]
    todo = [s for s, o in zip(srcs, objs) if force or _stale(o, [os.path.join(CSRC, s)] + HEADERS + [os.path.abspath(__file__)])]
    if todo:
        if verbose:
            print("compiling", todo, flush=True)
        with cf.ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as ex:
            list(ex.map(_compile, todo))
    if todo or _stale(LIB, objs):
        cmd = [NVCC] + ARCH + ["-shared", "-cudart", "static", "-o", LIB] + objs + ["-Xcompiler", "-pthread"]
        r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed: %s\n%s" % (" ".join(cmd), r.stdout[-4000:]))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
