"""Builds libncclx_b200.so IN-TREE with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libncclx_b200.so")
SOURCES = [os.path.join(CSRC, "ncclx_b200.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("common.cuh", "counts_kernel.cuh", "copy_kernel.cuh", "reduce_kernel.cuh", "dynamic_kernel.cuh", "topk_kernel.cuh", "fused_kernel.cuh", "probe_kernel.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "ncclx_b200.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "--ftz=false", "--prec-div=true",
              "--fmad=false"]


def nvcc() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    raise RuntimeError("nvcc not found")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *SOURCES]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


def build_variant(defines, out_path: str) -> str:
    """The same sources compiled with extra -D flags into `out_path` (never the default library).  Used by
    tests/test_zy_barrier_fallback.py for the -DXDEV_TEST_FORCE_BARRIER_TIMEOUT build; select the result with
    NCCLX_B200_LIB=<path>."""
    assert os.path.abspath(out_path) != LIB
    tmp = out_path + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc(), *NVCC_FLAGS, *defines, "-o", tmp, *SOURCES])
    os.replace(tmp, out_path)
    return out_path


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
