"""Build the cuFFT+cuRAND comparison step (compare/cufft_modelb.cu) into compare/libpss_cufft_compare.so.

Bench and test infrastructure only: the paper's kernel-per-arrow structure with library FFTs and library noise, timed
for context by bench.py, and the cuRAND Philox hook of pin P8.  It lives outside the product package and is never
loaded by paper_2405_02410_b200/.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cufft_modelb.cu")
LIB = os.path.join(HERE, "libpss_cufft_compare.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(SRC) > os.path.getmtime(LIB):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + ".tmp.%d" % os.getpid()
        subprocess.run([nvcc] + NVCC_FLAGS + ["-o", tmp, SRC, "-lcufft", "-lcurand"], check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
