"""Build libmd_b200.so (sm_100a) in-tree with nvcc.  `python -m paper_2003_14061_b200.build [--verbose]`."""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libmd_b200.so")
SOURCES = ["md_api.cu", "md_kernels.cu", "md_tile.cu", "md_sp.cu", "md_pushoff.cu", "md_peaks.cu", "md_rigid.cu", "md_noalloc.cu", "md_init.cpp"]
HEADERS = [os.path.join(CSRC, "md_types.h"), os.path.join(CSRC, "md_device.cuh"), os.path.join(CSRC, "md_rebuild.cuh"), os.path.join(CSRC, "md_init.h"), os.path.join(ROOT, "include", "md_b200.h")]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, extra_flags=()) -> str:
    if not force and not needs_build():
        return LIB
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "--shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
           "-I", os.path.join(ROOT, "include"), "-I", CSRC, "-o", LIB]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += list(extra_flags)                                    # tuning experiments, e.g. -DMD_FORCE_U=2
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    # python -m paper_2003_14061_b200.build [--verbose] [-- <extra nvcc flags>]
    extra = sys.argv[sys.argv.index("--") + 1:] if "--" in sys.argv else []
    print(build(force=True, verbose="--verbose" in sys.argv, extra_flags=extra))
