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


SANITIZED_LIB = os.path.join(HERE, "libmuon_oracle_asan.so")
SANITIZE_FLAGS = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]


def build(force: bool = False, sanitize: bool = False) -> str:
    """sanitize=True: the same source with AddressSanitizer and UndefinedBehaviorSanitizer as
    libmuon_oracle_asan.so; run the CPU tests against it with
        LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
        MUON_ORACLE_LIB=oracle/libmuon_oracle_asan.so python -m pytest tests -q -m "not gpu"
    (profiles/r2_sanitizers.md has the record)."""
    lib = SANITIZED_LIB if sanitize else LIB
    if (not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(SRC)):
        return lib
    tmp = lib + ".tmp.%d" % os.getpid()
    flags = [f for f in FLAGS if f != "-O2"] + SANITIZE_FLAGS if sanitize else FLAGS
    subprocess.check_call(["g++", *flags, SRC, "-o", tmp])
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    import sys
    print(build(force=True, sanitize="--sanitize" in sys.argv))
