"""Build `libfkconv.so` (the C-ABI library of include/fkconv.h) in-tree with nvcc for sm_100a.

    python -m paper_1909_10547_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU; the built .so is git-ignored but travels with the tree.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfkconv.so")
OBJDIR = os.path.join(HERE, "build")   # object files (git-ignored)
# translation units -> the files each one includes (a unit is recompiled when one of them changes)
UNITS = {
    "fk_api.cu": ["fk_api.cu", "fk_group.inl", "fk_common.cuh", "fk_fwd.cuh", "fk_vjp.cuh", "fk_gemm.cuh", "fk_gemm_ws.cuh",
                  "fk_vjp_fold.cuh", "fk_chi2.cuh", "fk_pack.cuh", "fk_tc32.h", "fk_sparse.cuh", "fk_dis_direct.cuh"],
    "fk_tc32.cu": ["fk_tc32.cu", "fk_tc32.h", "fk_common.cuh"],
}

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the FK convolution library cannot be built")


def _unit_stale(unit: str) -> bool:
    obj = os.path.join(OBJDIR, unit + ".o")
    if not os.path.exists(obj):
        return True
    t = os.path.getmtime(obj)
    deps = [os.path.join(CSRC, d) for d in UNITS[unit]] + [os.path.join(ROOT, "include", "fkconv.h"), os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def stale() -> bool:
    return not os.path.exists(LIB) or any(_unit_stale(u) for u in UNITS) or any(
        os.path.getmtime(os.path.join(OBJDIR, u + ".o")) > os.path.getmtime(LIB) for u in UNITS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compiles the stale translation units (in parallel) and links libfkconv.so."""
    if not force and not stale():
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    procs = []
    for unit in UNITS:
        if not force and not _unit_stale(unit):
            continue
        obj = os.path.join(OBJDIR, unit + ".o")
        cmd = [_nvcc(), *NVCC_FLAGS, "-c"]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += ["-o", obj + ".tmp", os.path.join(CSRC, unit)]
        procs.append((unit, obj, cmd, subprocess.Popen(cmd, cwd=CSRC)))
    for unit, obj, cmd, p in procs:
        if p.wait() != 0:
            raise subprocess.CalledProcessError(p.returncode, cmd)
        os.replace(obj + ".tmp", obj)
    tmp = LIB + ".tmp%d" % os.getpid()
    subprocess.check_call([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-o", tmp]
                          + [os.path.join(OBJDIR, u + ".o") for u in UNITS], cwd=CSRC)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
