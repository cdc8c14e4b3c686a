"""Compile the CPU oracle (oracle/opss.cpp) into oracle/libopss.so with g++.

TEST INFRASTRUCTURE: building the checker is not using it.  Called by
``__graft_entry__.build()`` and lazily by ``oracle/opss.py``.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "opss.cpp")
HDR = os.path.join(HERE, "opss.h")
LIB = os.path.join(HERE, "libopss.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in (SRC, HDR))


def build(force: bool = False) -> str:
    """OPSS_SANITIZE=1 builds with -fsanitize=address,undefined (run the pins with LD_PRELOAD=$(g++ -print-file-name=libasan.so))."""
    global LIB
    san = os.environ.get("OPSS_SANITIZE", "") not in ("", "0")
    if san:
        LIB = os.path.join(HERE, "libopss_san.so")
    if force or needs_build():
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-Wall", "-Wextra"] + (["-fsanitize=address,undefined", "-fno-omit-frame-pointer", "-g"] if san else []) + ["-o", tmp, SRC]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
