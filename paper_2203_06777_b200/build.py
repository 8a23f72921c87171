"""Build libdwf.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2203_06777_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so sits next to this file so that it travels with the
source tree (it is git-ignored, not gpurun-ignored).
"""
from __future__ import annotations

import concurrent.futures
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libdwf.so")
OBJDIR = os.path.join(HERE, "build")

# (source, object name, extra defines): dhop_staged.cu and dhop_staged64.cu are compiled once per kernel
# MODE so that the sets of template instances build in parallel
SOURCES = [*[("dhop_staged64.cu", f"dhop_staged64_m{m}.o", [f"-DDWF_STAGED64_MODE={m}"]) for m in range(5)],
           ("api.cu", "api.o", []), ("pack.cu", "pack.o", []), ("dhop.cu", "dhop.o", []), ("reduce.cu", "reduce.o", []),
           ("dhop_staged.cu", "dhop_staged_m0.o", ["-DDWF_STAGED_MODE=0"]),
           ("dhop_staged.cu", "dhop_staged_m1.o", ["-DDWF_STAGED_MODE=1"]),
           ("dhop_staged.cu", "dhop_staged_m2.o", ["-DDWF_STAGED_MODE=2"]),
           ("dhop_staged.cu", "dhop_staged_m3.o", ["-DDWF_STAGED_MODE=3"]),
           ("dhop_staged.cu", "dhop_staged_m4.o", ["-DDWF_STAGED_MODE=4"]),
           ("dhop_staged.cu", "dhop_staged_m5.o", ["-DDWF_STAGED_MODE=5"]),
           ("dhop_staged.cu", "dhop_staged_m6.o", ["-DDWF_STAGED_MODE=6"]),
           ("dhop_staged.cu", "dhop_staged_m7.o", ["-DDWF_STAGED_MODE=7"]),
           ("dwf5d.cu", "dwf5d.o", []), ("halo.cu", "halo.o", []), ("norm2_static.cu", "norm2_static.o", []), ("half.cu", "half.o", [])]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: cannot build libdwf.so")
    return exe


def _deps():
    out = [os.path.join(ROOT, "include", "dwf.h"), os.path.abspath(__file__)]
    for f in os.listdir(CSRC):
        out.append(os.path.join(CSRC, f))
    return out


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    nvcc = _nvcc()
    extra = ["-Xptxas", "-v"] if verbose else []

    def compile_one(item):
        src, objname, defines = item
        obj = os.path.join(OBJDIR, objname)
        cmd = [nvcc, *NVCC_FLAGS, *extra, *defines, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        return objname, obj, r

    with concurrent.futures.ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    objs = []
    for src, obj, r in results:
        if verbose or r.returncode:
            sys.stderr.write(f"--- {src}\n{r.stdout}{r.stderr}\n")
        if r.returncode:
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(obj)
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc, "-shared", "-o", tmp, *objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
