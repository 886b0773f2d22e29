"""SURVEY.md §8(c) pin P-1 on the GPU box: cuRAND's Philox4x32-10 (an implementation that shares nothing with this
repository) against the oracle's Philox and against the words the step loop draws (mt_debug_philox), for the counter
layout of DESIGN.md §3.0: key = (seed lo, seed hi), counter = (id lo, id hi, step, 0)."""
import ctypes
import os
import subprocess

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))
CASES = ((1, 0, 0), (1, 0, 1), (0x0123456789ABCDEF, 0xFFFFFFF0, 77), (2 ** 63 + 5, 2 ** 40 + 3, 4099),
         (0xFFFFFFFFFFFFFFFF, 2 ** 61, 0xFFFFFFFF))


def _oracle_blocks(oracle, seed, id_base, step, n):
    ids = np.uint64(id_base) + np.arange(n, dtype=np.uint64)
    ctr = np.zeros((n, 4), np.uint32)
    ctr[:, 0] = (ids & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    ctr[:, 1] = (ids >> np.uint64(32)).astype(np.uint32)
    ctr[:, 2] = step
    return oracle.philox4x32_10(ctr, np.array([seed & 0xFFFFFFFF, seed >> 32], np.uint32))


@pytest.fixture(scope="module")
def curand_pin(tmp_path_factory):
    """the device-API helper (tests/curand_pin.cu), compiled here with nvcc for sm_100a"""
    from paper_2512_10520_b200.build import _nvcc
    so = str(tmp_path_factory.mktemp("curand_pin") / "libcurand_pin.so")
    subprocess.run([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-shared", "-Xcompiler", "-fPIC",
                    "-o", so, os.path.join(HERE, "curand_pin.cu")], check=True)
    lib = ctypes.CDLL(so)
    lib.curand_philox_blocks.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_void_p]
    lib.curand_philox_blocks.restype = ctypes.c_int
    return lib


def test_philox_device_api(curand_pin, mt, oracle):
    """curand_init(seed, subsequence = step, offset = 4 id) + curand4 == the oracle's block == the step loop's block"""
    import torch
    b = mt.binding
    ctx = b.mt_create(0)
    try:
        n = 4096
        for seed, id_base, step in CASES:
            out = torch.zeros((n, 4), dtype=torch.int32, device="cuda")
            torch.cuda.synchronize()
            assert curand_pin.curand_philox_blocks(seed, id_base, step, n, out.data_ptr()) == 0
            theirs = out.cpu().numpy().view(np.uint32)
            assert np.array_equal(_oracle_blocks(oracle, seed, id_base, step, n), theirs), (seed, id_base, step)
            ours = b.mt_debug_philox(ctx, seed, id_base, step, n).cpu().numpy().view(np.uint32)
            assert np.array_equal(ours, theirs), (seed, id_base, step)
    finally:
        b.mt_destroy(ctx)


def test_philox_host_api(oracle):
    """libcurand's host generator (no code of ours on the device).  Its default ordering gives thread t of the generator
    subsequence t, i.e. the counter (0, 0, t, 0): block t of a request that starts at offset 0 is the block of muon 0 at
    step t (observed on this cuRAND, 10.3: block 1 of the stream is the block of counter (0, 0, 1, 0)).  Only the head of
    the request is compared, well below the generator's thread count."""
    import torch
    lib = None
    for name in ("libcurand.so.10", "/usr/local/cuda/lib64/libcurand.so.10", "libcurand.so"):
        try:
            lib = ctypes.CDLL(name)
            break
        except OSError:
            continue
    if lib is None:
        import glob
        import nvidia.curand
        lib = ctypes.CDLL(glob.glob(os.path.join(os.path.dirname(nvidia.curand.__file__), "lib", "libcurand.so*"))[0])
    gen = ctypes.c_void_p()
    assert lib.curandCreateGenerator(ctypes.byref(gen), 161) == 0          # CURAND_RNG_PSEUDO_PHILOX4_32_10
    try:
        n = 64
        out = torch.zeros(4 * n, dtype=torch.int32, device="cuda")
        for seed in (1, 0x0123456789ABCDEF, 2 ** 63 + 5):
            assert lib.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_uint64(seed)) == 0
            assert lib.curandSetGeneratorOffset(gen, ctypes.c_uint64(0)) == 0
            assert lib.curandGenerate(gen, ctypes.c_void_p(out.data_ptr()), ctypes.c_size_t(4 * n)) == 0
            torch.cuda.synchronize()
            theirs = out.cpu().numpy().view(np.uint32).reshape(n, 4)
            want = np.concatenate([_oracle_blocks(oracle, seed, 0, t, 1) for t in range(n)])
            assert np.array_equal(want, theirs), seed
    finally:
        lib.curandDestroyGenerator(gen)
