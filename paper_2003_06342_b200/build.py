"""Build the C-ABI shared library ``liblbm_b200.so`` in-tree with nvcc for sm_100a (cross-compiles without a GPU).

``python -m paper_2003_06342_b200.build`` or :func:`build` (used by ``__graft_entry__.build``).
The ptxas resource report (registers / spills per kernel) is written next to the library as ``ptxas.log``.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC_DIR = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblbm_b200.so")
SOURCES = ["lbm.cu", "halo.cu", "noalloc.cu", "finite.cu", "state.cu", "inst_2d995_f64.cu", "inst_2d995_f32.cu", "inst_2d999_f64.cu", "inst_2d999_f32.cu",
           "inst_3d_f64.cu", "inst_3d_f32.cu", "inst_3d15_f64.cu", "inst_3d15_f32.cu"]


def deps():
    """Every file the library is built from: all of csrc/ and the public header."""
    return sorted(glob.glob(os.path.join(SRC_DIR, "*.cu")) + glob.glob(os.path.join(SRC_DIR, "*.cuh")) +
                  glob.glob(os.path.join(SRC_DIR, "*.h"))) + [os.path.join(HERE, "..", "include", "lbm.h")]


NVCC_COMPILE = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xptxas", "-v",
                "-Xcompiler", "-fPIC", "-c"]
NVCC_LINK = ["-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in deps())


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every translation unit in parallel (one nvcc per unit), then link the shared library."""
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    procs = []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_COMPILE + ["-o", obj, src]
        procs.append((cmd, obj, subprocess.Popen(cmd, cwd=SRC_DIR, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    log, failed = [], False
    for cmd, obj, p in procs:
        out = p.communicate()[0]
        log.append(" ".join(cmd) + "\n" + out)
        failed = failed or p.returncode != 0
    if not failed:
        cmd = [nvcc] + NVCC_LINK + ["-o", LIB] + [o for _, o, _ in procs]
        r = subprocess.run(cmd, cwd=SRC_DIR, capture_output=True, text=True)
        log.append(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        failed = r.returncode != 0
    with open(os.path.join(HERE, "ptxas.log"), "w") as fh:
        fh.write("\n".join(log))
    if verbose or failed:
        sys.stderr.write("\n".join(log)[-6000:])
    if failed:
        raise RuntimeError("nvcc failed (see %s)" % os.path.join(HERE, "ptxas.log"))
    return LIB


if __name__ == "__main__":
    print(build(force=True))
