"""Build paper_2402_05240_b200/libmhd.so (the C-ABI CUDA library, include/mhd.h) in-tree.

nvcc cross-compiles for sm_100a without a GPU.  No fast-math: fp64 division and sqrt stay
IEEE; FMA contraction is nvcc's default.  Run `python -m paper_2402_05240_b200.build`.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmhd.so")
SOURCES = [os.path.join(CSRC, "mhd_api.cu"), os.path.join(CSRC, "mhd_peaks.cu"),
           os.path.join(CSRC, "mhd_unit.cu"), os.path.join(CSRC, "mhd_noalloc.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("mhd_device.cuh", "mhd_grid.cuh", "mhd_kernels.cuh", "mhd_math.cuh",
                                                   "mhd_stage.cuh")] + [
    os.path.join(ROOT, "include", "mhd.h")]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


PTXAS_LOG = ""


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def build(force: bool = False, verbose: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS)):
        return LIB
    cmd = [nvcc()] + NVCC_FLAGS + ["-o", LIB] + SOURCES
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or res.returncode:
        print(res.stdout)
    if res.returncode:
        raise RuntimeError("nvcc failed: %s" % " ".join(cmd))
    global PTXAS_LOG
    PTXAS_LOG = res.stdout   # registers / spills / shared memory per kernel (-Xptxas -v); nothing is written
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
