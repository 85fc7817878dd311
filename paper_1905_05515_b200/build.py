"""Build step of the CUDA library: nvcc -> paper_1905_05515_b200/libtpc_b200.so (in-tree, sm_100a only).

Run as `python -m paper_1905_05515_b200.build [--force]`; `__graft_entry__.build()` calls `build()`.
nvcc cross-compiles without a GPU.  -fmad=false: no FMA contraction anywhere in the library, so every fp32 product is rounded
before it is added, as the fp32 definition of the decision predicates requires (D-list); the fused
multiply-adds that reading A43 defines for the S5 transport / update are explicit __fmaf_rn calls in csrc/kalman.cuh.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libtpc_b200.so")
SO_CHECKED = os.path.join(HERE, "libtpc_b200_checked.so")   # same sources with -DTPC_CHECKED: bounds checks in the kernels (tests only)
SOURCES = ["tpc_abi.cu", "scan.cu", "k1_grid.cu", "k2_neighbours.cu", "k3_clean_start.cu", "k5_tracklets.cu", "k6_selector.cu", "k7_refit.cu", "k8_tube.cu", "k9_merge.cu", "k10_loopers.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-fmad=false", "-std=c++17",
              "-Xcompiler", "-fPIC", "-cudart", "shared"] + os.environ.get("TPC_NVCC_EXTRA", "").split()


def _nvcc() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    return "nvcc"


def _stale(so) -> bool:
    if not os.path.exists(so):
        return True
    t = os.path.getmtime(so)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "tpc.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def _build_one(so: str, extra: list, objdir: str, verbose: bool) -> None:
    os.makedirs(objdir, exist_ok=True)
    procs = []
    for s in SOURCES:
        cmd = [_nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, s), "-o",
                                                                                          os.path.join(objdir, s[:-3] + ".o")]
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for s, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode:
            sys.stderr.write(out)
        if p.returncode:
            raise RuntimeError(f"nvcc failed on {s}")
    cmd = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "shared", "-o", so] + \
          [os.path.join(objdir, s[:-3] + ".o") for s in SOURCES] + ["-Xlinker", "-rpath=/usr/local/cuda/lib64"]
    subprocess.check_call(cmd)


def build(force: bool = False, verbose: bool = False) -> str:
    """The product library, and beside it the checked build (same sources, -DTPC_CHECKED: bounds checks in the kernels) that
    tests/test_gpu_checked.py runs; the product never loads the checked build."""
    if force or _stale(SO):
        _build_one(SO, [], os.path.join(HERE, "build"), verbose)
    if force or _stale(SO_CHECKED):
        _build_one(SO_CHECKED, ["-DTPC_CHECKED"], os.path.join(HERE, "build", "checked"), False)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
