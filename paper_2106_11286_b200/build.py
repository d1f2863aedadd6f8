"""Build libhb.so (the C-ABI library of include/hb.h) in-tree with nvcc for sm_100a.

    python -m paper_2106_11286_b200.build [--force]

The .so is git-ignored but travels with the gpurun snapshot.  No JIT, no torch
extension machinery: the library has no torch types in its interface.
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libhb.so")
SOURCES = ["hb_api.cpp", "hb_lattice.cpp", "hb_kernels.cu", "hb_bravais.cu", "hb_bravais_ws.cu", "hb_ell.cu", "hb_sc_ws.cu", "hb_probe.cu", "hb_noalloc.cu"]
HEADERS = ["hb_internal.h", "hb_device.cuh", "hb_ws.cuh", "hb_bravais_geo.cuh", os.path.join("..", "..", "include", "hb.h"),
           os.path.join("..", "..", "include", "hb_noalloc.h"), os.path.join("..", "..", "include", "hb_diag.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-fmad=false",           # the arithmetic contract spells out every fused multiply-add
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "--threads", "0",
]


def nvcc():
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA extension cannot be built")
    return exe


def stale():
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not stale():
        return SO
    tmp = SO + ".tmp%d" % os.getpid()
    cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-x", "cu"] + [os.path.join(CSRC, f) for f in SOURCES] + ["-o", tmp]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stderr)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
