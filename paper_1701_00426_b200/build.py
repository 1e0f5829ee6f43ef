"""Build liblqcd_b200.so (in-tree) from csrc/*.cu with nvcc for sm_100a.

nvcc cross-compiles without a GPU, so this also runs on the CPU-only build box
(__graft_entry__.build()).  Objects go to csrc/build/ (git-ignored); the .so sits next to
this file so that it travels to the GPU box with the repository snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "liblqcd_b200.so")
SOURCES = ["api.cu", "pack.cu", "dslash.cu", "solver.cu", "host.cu", "force.cu", "staples.cu", "diag.cu", "peer.cu", "noalloc.cu", "dslash_multi.cu"]
HEADERS = ["common.cuh", "reduce.cuh", "su3.cuh", "peer.cuh", os.path.join("..", "..", "include", "lqcd.h"),
           os.path.join("..", "..", "include", "lqcd_diag.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src: str) -> str:
    obj = os.path.join(OBJ, src.replace(".cu", ".o"))
    deps = [os.path.join(CSRC, src)] + [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]
    if _stale(obj, deps):
        log = obj + ".log"
        with open(log, "w") as f:
            r = subprocess.run([NVCC] + FLAGS + ["-c", os.path.join(CSRC, src), "-o", obj],
                               stdout=f, stderr=subprocess.STDOUT)
        if r.returncode:
            sys.stderr.write(open(log).read())
            raise RuntimeError(f"nvcc failed on {src}")
    return obj


def build(force: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    if force:
        for f in os.listdir(OBJ):
            os.remove(os.path.join(OBJ, f))
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(_compile, SOURCES))
    if _stale(LIB, objs):
        subprocess.run([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs,
                       check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
