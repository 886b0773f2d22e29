"""Pins for the oracle's Philox4x32-10 (pin P-1)."""
import os

import numpy as np
import pytest
from scipy import stats


def test_philox_matches_triton_interpreter(oracle):
    """Independent implementation: Triton's tl.philox run by Triton's CPU interpreter."""
    os.environ["TRITON_INTERPRET"] = "1"
    try:
        import torch
        import triton
        import triton.language as tl
    except Exception as e:  # pragma: no cover
        pytest.skip("triton not importable: %r" % (e,))

    @triton.jit
    def kern(out, seed, c0p, c1p, c2p, c3p, n: tl.constexpr):
        i = tl.arange(0, n)
        r0, r1, r2, r3 = tl.philox(seed, tl.load(c0p + i), tl.load(c1p + i), tl.load(c2p + i), tl.load(c3p + i), 10)
        tl.store(out + i, r0)
        tl.store(out + n + i, r1)
        tl.store(out + 2 * n + i, r2)
        tl.store(out + 3 * n + i, r3)

    n = 64
    rng = np.random.default_rng(7)
    ctr = rng.integers(0, 2 ** 32, (n, 4), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0
    ctr[1] = 0xFFFFFFFF
    for seed in (0, 1, 0x1ABCDEF012345678, 0x7FFFFFFFFFFFFFFF):
        cols = [torch.from_numpy(ctr[:, j].copy().view(np.int32)) for j in range(4)]
        out = torch.zeros(4 * n, dtype=torch.int32)
        try:
            kern[(1,)](out, seed, *cols, n=n)
        except Exception as e:  # pragma: no cover
            pytest.skip("triton interpreter unavailable: %r" % (e,))
        theirs = out.numpy().view(np.uint32).reshape(4, n).T
        ours = oracle.philox4x32_10(ctr, np.array([seed & 0xFFFFFFFF, seed >> 32], np.uint32))
        assert np.array_equal(ours, theirs)


def test_muon_words_counter_layout(oracle):
    """key = (seed lo, seed hi); counter = (id lo, id hi, step, 0)  -- DESIGN.md §3.0"""
    seed, mid, step = 0x0123456789ABCDEF, 0x1122334455667788, 4242
    w = oracle.muon_words(seed, mid, step)
    ref = oracle.philox4x32_10(np.array([[mid & 0xFFFFFFFF, mid >> 32, step, 0]], np.uint32),
                               np.array([seed & 0xFFFFFFFF, seed >> 32], np.uint32))[0]
    assert np.array_equal(w, ref)
    # every coordinate of (seed, id, step) changes the block
    assert not np.array_equal(w, oracle.muon_words(seed + 1, mid, step))
    assert not np.array_equal(w, oracle.muon_words(seed, mid + 1, step))
    assert not np.array_equal(w, oracle.muon_words(seed, mid + (1 << 32), step))
    assert not np.array_equal(w, oracle.muon_words(seed, mid, step + 1))


def test_philox_words_uniform(oracle):
    n = 200_000
    ctr = np.zeros((n, 4), np.uint32)
    ctr[:, 0] = np.arange(n)          # consecutive muon ids
    ctr[:, 2] = 17
    w = oracle.philox4x32_10(ctr, np.array([1, 0], np.uint32))
    for j in range(4):
        top = np.bincount(w[:, j] >> 24, minlength=256)
        low = np.bincount(w[:, j] & 0xFF, minlength=256)
        assert stats.chisquare(top).pvalue > 1e-4
        assert stats.chisquare(low).pvalue > 1e-4
    u = (w >> 8).astype(np.float32) * np.float32(2.0 ** -24)
    assert u.max() < 1.0 and u.min() >= 0.0
    # consecutive ids / consecutive steps are uncorrelated
    assert abs(np.corrcoef(u[:-1, 0], u[1:, 0])[0, 1]) < 0.01
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.01
