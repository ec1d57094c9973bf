"""Build oracle/liblgt_oracle.so with g++ (no CUDA, no torch).

TEST INFRASTRUCTURE: the oracle is the parity reference and the timed CPU baseline,
never part of the product path.  `python -m oracle.build` or `oracle.build.build()`.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lgt_oracle.cpp")
HDR = os.path.join(HERE, "lgt_oracle.h")
LIB = os.path.join(HERE, "liblgt_oracle.so")

# -fcx-limited-range: plain (ac-bd, ad+bc) complex products without the C99 Annex G
# inf/nan recovery call; finite results are identical, the loops are several times faster.
FLAGS = ["-O2", "-std=c++17", "-fopenmp", "-fcx-limited-range", "-fPIC", "-shared", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    newest_src = max(os.path.getmtime(SRC), os.path.getmtime(HDR), os.path.getmtime(__file__))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest_src:
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["g++", *FLAGS, "-o", tmp, SRC])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
