"""Build libmuon_transport.so (the C-ABI library) in-tree with nvcc for sm_100a.

    python -m paper_2512_10520_b200.build [--force]

nvcc cross-compiles without a GPU.  No -use_fast_math and no FMA contraction: the kernels spell every
rounding themselves (csrc/mt_step.cuh), -fmad=false is belt and braces.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libmuon_transport.so")
SOURCES = ["mt_lib.cu", "mt_kernels.cu"]
DEPS = SOURCES + ["mt_step.cuh", "mt_params.h", "mt_launch.h"]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-fmad=false",
              "-Xcompiler", "-fPIC,-Wall", "-shared", "-Xptxas", "-v"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False, defines=()) -> str:
    """`defines`: extra -D macros (e.g. MT_MIN_BLOCKS=4, MT_MAX_THREADS=128) for tuning experiments."""
    deps = [os.path.join(CSRC, d) for d in DEPS] + [os.path.join(INCLUDE, "muon_transport.h"), __file__]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc(), *NVCC_FLAGS, *["-D" + d for d in defines], "-I", INCLUDE, "-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout)
        raise RuntimeError("nvcc failed building libmuon_transport.so")
    if verbose:
        print(res.stdout)
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    with open(os.path.join(HERE, "build", "ptxas.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stdout)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv or any(a.startswith("-D") for a in sys.argv), verbose="--quiet" not in sys.argv,
                defines=[a[2:] for a in sys.argv if a.startswith("-D")]))
