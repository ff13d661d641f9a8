"""Builds paper_2606_09551_b200/libfusefss.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libfusefss.so")
import glob

SOURCES = ["libfusefss.cu", "compile.cpp"]


def deps():
    """every file the library is built from: all of csrc/ plus the public header"""
    return sorted(glob.glob(os.path.join(_CSRC, "*"))) + [os.path.join(_HERE, "..", "include", "fusefss.h")]


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    newest = max(os.path.getmtime(d) for d in deps())
    flags_file, want = LIB + ".flags", " ".join(extra)
    have = open(flags_file).read() if os.path.exists(flags_file) else ""
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest and have == want:   # up to date AND built with these switches
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
           "-Xcompiler", "-fPIC,-Wall", "--expt-relaxed-constexpr", "-split-compile", "0", "-o", LIB]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += list(extra) + [os.path.join(_CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    with open(flags_file, "w") as f:
        f.write(want)
    return LIB


if __name__ == "__main__":
    # python paper_2606_09551_b200/build.py [-v] [-DNAME=VALUE ...]   (the -D switches: tuning macros such as FFS_SP_THREADS,
    # FFS_P3_THREADS, FFS_SP_NP_BIG, FFS_SP_L2HINT -- see profiles/r2d_eval_sp_sweep.md; a plain build() restores the defaults)
    import sys
    print(build(force=True, verbose="-v" in sys.argv, extra=[a for a in sys.argv[1:] if a.startswith("-D")]))
