"""Builds libtpc_cf.so (the C-ABI library of include/tpc_cf.h, include/tpc_ec.h and include/tpc_fe.h) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  The built .so is git-ignored but travels with the snapshot to the GPU box.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
SO = os.path.join(_HERE, "libtpc_cf.so")
import glob

SOURCES = ["tpc_cf_api.cu", "tpc_cf_general.cu", "tpc_cf_fused.cu", "tpc_cf_blocks.cu", "tpc_cf_pairs.cu", "tpc_cf_sort.cu",
           "tpc_cf_compact.cu", "tpc_cf_share.cu", "tpc_ec.cu", "tpc_fe.cu"]
HEADERS = sorted(glob.glob(os.path.join(CSRC, "*.cuh")) +
                 glob.glob(os.path.join(os.path.dirname(_HERE), "include", "*.h")))
EXTRA = os.environ.get("TPC_CF_NVCC_EXTRA", "").split()
NVCC_FLAGS = EXTRA + ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "-ldl"]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def stale():
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not stale():
        return SO
    tmp = SO + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force=True, verbose=True))
