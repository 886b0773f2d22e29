"""Build libmuon_transport.so (the C-ABI library) and libmuon_probes.so (the measurement probes of include/muon_probes.h,
which only bench.py and the tests load) in-tree with nvcc for sm_100a.

    python -m paper_2512_10520_b200.build [--force]

nvcc cross-compiles without a GPU.  No -use_fast_math and no FMA contraction: the kernels spell every
rounding themselves (csrc/mt_step.cuh), -fmad=false is belt and braces.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libmuon_transport.so")
SOURCES = ["mt_lib.cu", "mt_kernels.cu", "mt_inst_regions.cu", "mt_inst_poly.cu", "mt_inst_voxel_a.cu",
           "mt_inst_voxel_b.cu", "mt_inst_lean.cu"]
# the measurement probes (include/muon_probes.h) are a library of their own: bench.py and tests load it, the product does not
PROBES_LIB = os.path.join(HERE, "libmuon_probes.so")
PROBE_SOURCES = ["mt_probe.cu", "mt_probe_field.cu"]
DEPS = SOURCES + PROBE_SOURCES + ["mt_kernels.cuh", "mt_step.cuh", "mt_params.h", "mt_launch.h"]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-fmad=false",
              "-Xcompiler", "-fPIC,-Wall", "-Xptxas", "-v"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


CHECKED_LIB = os.path.join(HERE, "libmuon_transport_checked.so")


def build(force: bool = False, verbose: bool = False, defines=(), checked: bool = False) -> str:
    """Compile the translation units in parallel (the kernel instantiations are split over several so that this takes
    about a minute on 8 cores), then link.  `defines`: extra -D macros (e.g. MT_MAX_THREADS=1024) for tuning experiments.
    checked=True builds libmuon_transport_checked.so with -DMT_CHECKED: the same kernels with every global-array index
    bounds-checked (csrc/mt_params.h: MT_CHECK); load it through MUON_TRANSPORT_LIB (tests/test_gpu_checked.py)."""
    LIB = CHECKED_LIB if checked else globals()["LIB"]
    defines = tuple(defines) + (("MT_CHECKED",) if checked else ())
    deps = [os.path.join(CSRC, d) for d in DEPS] + [os.path.join(INCLUDE, "muon_transport.h"),
                                                     os.path.join(INCLUDE, "muon_probes.h"), __file__]
    targets = [LIB] if checked else [LIB, PROBES_LIB]
    if not force and all(os.path.exists(t) and all(os.path.getmtime(t) >= os.path.getmtime(d) for d in deps) for t in targets):
        return LIB
    sources = SOURCES if checked else SOURCES + PROBE_SOURCES
    bdir = os.path.join(HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    tag = ".%d%s" % (os.getpid(), ".chk" if checked else "")
    base = [_nvcc(), *NVCC_FLAGS, *["-D" + d for d in defines], "-I", INCLUDE]

    def compile_one(src):
        obj = os.path.join(bdir, src[:-3] + tag + ".o")
        cmd = base + ["-c", os.path.join(CSRC, src), "-o", obj]
        res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        return obj, cmd, res

    with ThreadPoolExecutor(max_workers=min(len(sources), os.cpu_count() or 1)) as pool:
        done = list(pool.map(compile_one, sources))
    log = []
    objs = []
    probe_objs = []
    try:
        for obj, cmd, res in done:
            log.append(" ".join(cmd) + "\n" + res.stdout)
            (probe_objs if os.path.basename(cmd[-3]) in PROBE_SOURCES else objs).append(obj)
            if res.returncode != 0:
                sys.stderr.write(res.stdout)
                raise RuntimeError("nvcc failed compiling " + cmd[-3])
        tmp = LIB + ".tmp" + tag
        link = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp] + objs
        res = subprocess.run(link, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        log.append(" ".join(link) + "\n" + res.stdout)
        if res.returncode != 0:
            sys.stderr.write(res.stdout)
            raise RuntimeError("nvcc failed linking libmuon_transport.so")
        os.replace(tmp, LIB)
        if probe_objs:
            tmp = PROBES_LIB + ".tmp" + tag
            link = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp] + probe_objs
            res = subprocess.run(link, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
            log.append(" ".join(link) + "\n" + res.stdout)
            if res.returncode != 0:
                sys.stderr.write(res.stdout)
                raise RuntimeError("nvcc failed linking libmuon_probes.so")
            os.replace(tmp, PROBES_LIB)
    finally:
        for obj, _, _ in done:                    # every object this build wrote, also after a failed compile
            if os.path.exists(obj):
                os.remove(obj)
        with open(os.path.join(bdir, "ptxas_checked.log" if checked else "ptxas.log"), "w") as f:
            f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv or any(a.startswith("-D") for a in sys.argv), verbose="--quiet" not in sys.argv,
                defines=[a[2:] for a in sys.argv if a.startswith("-D")], checked="--checked" in sys.argv))
