"""Build libhlb.so in-tree with nvcc for sm_100a (no JIT cache, the .so travels with the repo)."""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
# HLB_LIB_PATH (tuning experiments only): build / load another copy of the library, e.g. one made
# with HLB_EXTRA_NVCC_FLAGS, so that several variants can be compared in one GPU session
LIB_PATH = os.environ.get("HLB_LIB_PATH") or os.path.join(HERE, "libhlb.so")
SOURCES = ["api.cu", "kernels.cu", "render.cu", "preprocess.cpp"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "--threads", "4", "--shared", "-Xcompiler", "-fPIC,-O3,-Wall,-pthread", "-cudart", "static",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libhlb.so cannot be built")


def _deps():
    out = [os.path.join(INCLUDE, "hlb.h"), os.path.abspath(__file__)]
    for f in sorted(os.listdir(CSRC)):
        out.append(os.path.join(CSRC, f))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(f) for f in _deps())
    if not force and os.path.exists(LIB_PATH) and \
            (os.path.getmtime(LIB_PATH) >= newest or os.environ.get("HLB_NO_REBUILD") == "1"):
        return LIB_PATH   # (HLB_NO_REBUILD: tuning runs that compare libraries built from other sources)
    tmp = LIB_PATH + f".tmp{os.getpid()}"
    extra = os.environ.get("HLB_EXTRA_NVCC_FLAGS", "").split()   # tuning experiments only
    cmd = [_nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + \
        ["-I", INCLUDE, "-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libhlb.so")
    os.replace(tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
