"""Build the C-ABI shared library ``liblbm_b200.so`` in-tree with nvcc for sm_100a (cross-compiles without a GPU).

``python -m paper_2003_06342_b200.build`` or :func:`build` (used by ``__graft_entry__.build``).
The ptxas resource report (registers / spills per kernel) is written next to the library as ``ptxas.log``.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC_DIR = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblbm_b200.so")
SOURCES = ["lbm.cu"]
DEPS = ["lbm.cu", "kernels.cuh", "k_phi.cuh", "k_main.cuh", "k_main_tma.cuh", "lattices.cuh", os.path.join("..", "..", "include", "lbm.h")]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xptxas", "-v",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(SRC_DIR, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", LIB] + SOURCES
    r = subprocess.run(cmd, cwd=SRC_DIR, capture_output=True, text=True)
    with open(os.path.join(HERE, "ptxas.log"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed (see %s)" % os.path.join(HERE, "ptxas.log"))
    return LIB


if __name__ == "__main__":
    print(build(force=True))
