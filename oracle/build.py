"""Build oracle/libmuon_oracle.so with g++ (TEST INFRASTRUCTURE ONLY; see muon_oracle.cpp header).

-ffp-contract=off keeps every float32 operation a single rounding in the written order;
fused multiply-adds happen only where the source calls std::fma.  -march=x86-64-v3 gives a hardware
fma without tying the binary to the build machine.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "muon_oracle.cpp")
LIB = os.path.join(HERE, "libmuon_oracle.so")

FLAGS = ["-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
         "-march=x86-64-v3", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["g++", *FLAGS, SRC, "-o", tmp])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
