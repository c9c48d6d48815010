"""Build paper_2508_21208_b200/libdgswem.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

Flags that matter: -fmad=false and host -ffp-contract=off (the compilers contract nothing by
themselves -- fused multiply-adds are the explicit fma() calls of the canonical arithmetic -- so results are reproducible bit
for bit against the specification), -lineinfo (ncu source page).  csrc/dgswem.cu compiles kernels and host code twice (fp64, fp32);
csrc/dgswem_static.cu (the allocation-free nodal output) is linked into the same library."""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
SRC = PKG / "csrc" / "dgswem.cu"
SRC_STATIC = PKG / "csrc" / "dgswem_static.cu"   # dgswem_nodal_static: own translation unit, own file-scope scratch
DEPS = [SRC, SRC_STATIC, PKG / "csrc" / "dgswem_kernels.cuh", PKG / "csrc" / "dgswem_impl.inl", ROOT / "include" / "dgswem.h"]
LIB = PKG / "libdgswem.so"

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-fmad=false", "-split-compile", "0",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-O2", "-shared"]


def nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and LIB.exists() and LIB.stat().st_mtime >= max(d.stat().st_mtime for d in DEPS):
        return LIB
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    extra = os.environ.get("DGSWEM_NVCC_EXTRA", "").split()   # tuning sweeps: e.g. -DDGK_STAGE_MINB=4
    cmd = [nvcc(), *NVCC_FLAGS, *extra, "-I", str(ROOT / "include"), "-I", str(PKG / "csrc"), "-o", str(tmp), str(SRC), str(SRC_STATIC)]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    build(force=True, verbose="-v" in sys.argv)
    print(LIB)
