"""Build libetics.so (CUDA kernels + C ABI) in-tree for sm_100a.

    python -m paper_1406_4254_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU (about two minutes from scratch on 8 cores).  Objects are cached under paper_1406_4254_b200/build/ by mtime; the shared
library lands next to this file (git-ignored, but it travels to the GPU box with the tree).
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libetics.so")
# (source, object stem, extra flags).  mex.cu is compiled in four parts (ETICS_MEX_PART: sort + lmax <= 6 | 7-8 | 9 | 10):
# its template instances dominate the build and the parts compile in parallel.
SOURCES = [("etics_api.cu", "etics_api", []), ("scf.cu", "scf", []), ("probe.cu", "probe", []), ("mex_sort.cu", "mex_sort", []),
           ("stepper.cu", "stepper", []), ("scf_f32.cu", "scf_f32", []),
           ("scf_static.cu", "scf_static", [])] + \
          [("mex.cu", f"mex_p{k}", [f"-DETICS_MEX_PART={k}"]) for k in range(4)]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + os.environ.get("ETICS_NVCC_EXTRA", "").split()


def _deps_mtime() -> float:
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hdrs.append(os.path.join(os.path.dirname(HERE), "include", "etics.h"))
    return max(os.path.getmtime(h) for h in hdrs)


def _compile(item, force: bool, verbose: bool) -> str:
    src, stem, extra = item
    s = os.path.join(CSRC, src)
    o = os.path.join(OBJ, stem + ".o")
    if not force and os.path.exists(o) and os.path.getmtime(o) >= max(os.path.getmtime(s), _deps_mtime()):
        return o
    r = subprocess.run([NVCC, *FLAGS, *extra, "-c", s, "-o", o], capture_output=True, text=True)
    log = os.path.join(OBJ, stem + ".ptxas.log")
    with open(log, "w") as f:
        f.write(r.stderr)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}")
    return o


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(lambda s: _compile(s, force, verbose), SOURCES))
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        subprocess.run([NVCC, "-shared", "-o", LIB + ".tmp", *objs, "-lcudart"], check=True)
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
