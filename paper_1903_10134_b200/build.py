"""Builds libmdpd_b200.so (hand-written CUDA for sm_100a + the C-ABI of include/mdpd.h) in-tree with nvcc."""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
SRC = [os.path.join(PKG, "csrc", "mdpd_b200.cu")]
HDR = [os.path.join(ROOT, "include", "mdpd.h")]
LIB = os.path.join(PKG, "libmdpd_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "static",
    "-I", os.path.join(ROOT, "include"),
]


FLAGS_FILE = LIB + ".flags"   # the -D set the library on disk was built with (one line; "" = the plain build)


def flags_string(defines=()) -> str:
    """Canonical form of a -D set: sorted, comma-joined; also compiled into the library (mdpd_build_flags())."""
    return ",".join(sorted(set(defines)))


def built_flags():
    try:
        with open(FLAGS_FILE) as f:
            return f.read().strip()
    except OSError:
        return None


def needs_build(defines=()) -> bool:
    """Stale if a source is newer than the library OR the library on disk was built with another -D set (so a
    -DMDPD_CHECKS or -DMDPD_FIRST_TILE measurement build is never silently reused by the tests or bench.py, nor the
    plain build by a checks run)."""
    if not os.path.exists(LIB):
        return True
    if built_flags() != flags_string(defines):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SRC + HDR + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False, defines=()) -> str:
    """defines: extra -D options, e.g. ("-DMDPD_CHECKS",) for the build with the kernels' own bounds checks."""
    if force or needs_build(defines):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + f".tmp{os.getpid()}"
        tag = '-DMDPD_BUILD_FLAGS="%s"' % flags_string(defines)
        cmd = [nvcc] + NVCC_FLAGS + list(defines) + [tag] + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SRC
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
        with open(FLAGS_FILE, "w") as f:
            f.write(flags_string(defines) + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, defines=[a for a in sys.argv[1:] if a.startswith("-D")]))
