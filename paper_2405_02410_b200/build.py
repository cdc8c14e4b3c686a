"""Compile the CUDA product (csrc/pss.cu) into paper_2405_02410_b200/libpss.so for sm_100a.

In-tree build with nvcc (cross-compiles without a GPU); the .so travels to the GPU box with the
repository snapshot.  Called by ``__graft_entry__.build()`` and lazily by ``binding.lib()``.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libpss.so")
SOURCES = [os.path.join(CSRC, "pss.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in
                  ("pss_program.h", "pss_fft.cuh", "pss_pointwise.cuh", "pss_kernels.cuh", "pss_fused2d.cuh", "pss_persist2d.cuh")] + \
    [os.path.join(INCLUDE, "pss.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in DEPS if os.path.exists(p))


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = [nvcc] + NVCC_FLAGS + os.environ.get("PSS_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else []) + ["-I", INCLUDE, "-o", tmp] + SOURCES
        subprocess.run(cmd, check=True, cwd=CSRC)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
