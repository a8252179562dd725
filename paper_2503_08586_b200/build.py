"""Build libtinylens.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2503_08586_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library links the CUDA runtime statically, so it
loads on a machine without libcudart (compute calls then return TL_ECUDA).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtinylens.so")
SOURCES = [os.path.join(CSRC, f) for f in ("tinylens.cu", "tl_inst_fused.cu", "tl_inst_split.cu", "tl_inst_lin.cu",
                                           "tl_inst_epl.cu", "tl_inst_epl_lin.cu", "tl_inst_serve.cu", "tl_peaks.cu")]
HEADERS = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))) + \
          [os.path.join(os.path.dirname(HERE), "include", "tinylens.h")]

NVCC_COMPILE = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
]
NVCC_LINK = ["-gencode", "arch=compute_100a,code=sm_100a", "--shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    # the translation units are independent (no relocatable device code): compile them in
    # parallel, then link one shared library
    bdir = os.path.join(HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    procs, objs, log = [], [], []
    for src in SOURCES:
        obj = os.path.join(bdir, os.path.basename(src)[:-3] + ".%d.o" % os.getpid())
        cmd = [nvcc_path()] + NVCC_COMPILE + ["-c", "-o", obj, src]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    failed = None
    for cmd, p in procs:
        out, _ = p.communicate()
        log.append(" ".join(cmd) + "\n" + out)
        if p.returncode != 0 and failed is None:
            failed = (cmd, out)
    tmp = LIB + ".tmp.%d" % os.getpid()
    if failed is None:
        cmd = [nvcc_path()] + NVCC_LINK + ["-o", tmp] + objs
        proc = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        log.append(" ".join(cmd) + "\n" + proc.stdout)
        if proc.returncode != 0:
            failed = (cmd, proc.stdout)
    for o in objs:
        if os.path.exists(o):
            os.remove(o)
    if failed is not None:
        if os.path.exists(tmp):
            os.remove(tmp)
        raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(failed[0]), failed[1]))
    os.replace(tmp, LIB)
    with open(os.path.join(HERE, "build.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
