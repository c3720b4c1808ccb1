"""Build step: compiles csrc/*.cu into libdualip_b200.so (in-tree) for sm_100a with nvcc.

Run as `python -m paper_2606_07777_b200.build` or through `__graft_entry__.build()`.  nvcc cross-compiles
without a GPU.  The .so is git-ignored but travels to the GPU box with the working tree.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdualip_b200.so")
SOURCES = ["dualip_api.cu", "dualip_tma_wx0.cu", "dualip_tma_wx1.cu", "dualip_static.cu"]   # compiled in parallel, then linked
HEADERS = ["dualip_kernels.cuh", "dualip_grad_tma.cuh", "dualip_csc.cuh", "dualip_long.cuh", os.path.join("..", "..", "include", "dualip.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC,-O2,-Wall"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _compile_and_link(out: str, flags: list, log=None) -> None:
    """One nvcc -c per source, all at once (the template instantiations dominate the build time), then one link."""
    import tempfile
    with tempfile.TemporaryDirectory() as td:
        objs, procs = [], []
        for src in SOURCES:
            obj = os.path.join(td, src.replace(".cu", ".o"))
            objs.append(obj)
            procs.append(subprocess.Popen([_nvcc()] + flags + ["-c", "-o", obj, os.path.join(CSRC, src)],
                                          stdout=log, stderr=subprocess.STDOUT if log else None))
        rcs = [pr.wait() for pr in procs]
        if any(rcs):
            raise subprocess.CalledProcessError(max(rcs), "nvcc -c")
        subprocess.check_call([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", out] + objs)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    flags = list(NVCC_FLAGS)
    if verbose:
        flags += ["-Xptxas", "-v"]
    tmp = LIB + f".{os.getpid()}.tmp"
    _compile_and_link(tmp, flags)
    os.replace(tmp, LIB)
    return LIB


CHECKED_LIB = os.path.join(HERE, "libdualip_b200_checked.so")


def build_checked(force: bool = False) -> str:
    """The -DDUALIP_CHECKED variant (in-kernel bounds assertions, dualip_info.checks_failed) next to the product library;
    tests/test_gpu_checked_build.py loads it.  Not used by anything else."""
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    if force or not os.path.exists(CHECKED_LIB) or any(os.path.getmtime(d) > os.path.getmtime(CHECKED_LIB) for d in deps):
        tmp = CHECKED_LIB + f".{os.getpid()}.tmp"
        _compile_and_link(tmp, NVCC_FLAGS + ["-DDUALIP_CHECKED=1"])
        os.replace(tmp, CHECKED_LIB)
    return CHECKED_LIB


if __name__ == "__main__":
    if "--checked" in sys.argv:
        print(build_checked(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
