"""Pins for the oracle's alias-table construction and draw (P-2, P-3)."""
import numpy as np
import pytest
from scipy import stats


def implied_pmf(prob, alias):
    """Mass each outcome receives from the N equiprobable cells (the alias-method identity)."""
    N = len(prob)
    pmf = np.zeros(N)
    for k in range(N):
        pmf[k] += float(prob[k]) / N
        pmf[int(alias[k])] += (1.0 - float(prob[k])) / N
    return pmf


@pytest.mark.parametrize("N", [1, 2, 3, 7, 64, 128, 1000, 1024])
def test_build_conserves_mass(oracle, N):
    rng = np.random.default_rng(N)
    for trial in range(5):
        counts = rng.gamma(0.3, 1.0, N).astype(np.float32)
        if N > 3:
            counts[rng.integers(0, N, N // 4)] = 0.0          # empty cells
        if counts.sum() == 0:
            counts[0] = 1
        prob, alias = oracle.build_alias(counts)
        assert alias.max() < N and prob.min() >= 0.0 and prob.max() <= 1.0
        want = counts.astype(np.float64) / counts.astype(np.float64).sum()
        assert np.abs(implied_pmf(prob, alias) - want).max() < 1e-6
        # a cell with zero weight is never returned as a primary
        assert np.all(prob[counts == 0] == 0.0)


def test_build_special_cases(oracle):
    prob, alias = oracle.build_alias(np.full(16, 3.0, np.float32))         # uniform: every cell keeps itself
    assert np.all(prob == 1.0) and np.array_equal(alias, np.arange(16))
    prob, alias = oracle.build_alias(np.array([0, 0, 5, 0], np.float32))   # delta: everything lands on 2
    assert np.allclose(implied_pmf(prob, alias), [0, 0, 1, 0])
    with pytest.raises(ValueError):
        oracle.build_alias(np.zeros(8, np.float32))
    with pytest.raises(ValueError):
        oracle.build_alias(np.array([1, -1, 1], np.float32))


def test_build_batch_is_per_table(oracle):
    rng = np.random.default_rng(3)
    counts = rng.random((3, 5, 32)).astype(np.float32)
    prob, alias = oracle.build_alias(counts)
    p1, a1 = oracle.build_alias(counts[2, 4])
    assert np.array_equal(prob[2, 4], p1) and np.array_equal(alias[2, 4], a1)


def test_draw_exact_enumeration_tiny_table(oracle):
    """Brute force over ALL 2^32 words: the outcome frequencies are the pmf (to the 2^-24 grid of u)."""
    counts = np.array([5, 1, 0, 2, 7], np.float32)
    prob, alias = oracle.build_alias(counts)
    got = oracle.alias_enumerate(prob, alias).astype(np.float64) / 2.0 ** 32
    want = counts / counts.sum()
    assert got[2] == 0.0
    assert np.abs(got - want).max() < 2.0 ** -23


def test_draw_edge_words(oracle):
    counts = np.array([1, 3, 2, 2], np.float32)
    prob, alias = oracle.build_alias(counts)
    N = 4
    # word 0 -> cell 0, u = 0 (accept unless prob is 0); word 0xFFFFFFFF -> last cell, u just below 1
    cells = oracle.alias_draw(prob, alias, np.array([0, 0xFFFFFFFF], np.uint32))
    assert cells[0] == (0 if prob[0] > 0 else alias[0])
    k = (0xFFFFFFFF * N) >> 32
    u_last = np.float32((((0xFFFFFFFF * N) & 0xFFFFFFFF) >> 8) * 2.0 ** -24)
    assert cells[1] == (k if u_last < prob[k] else alias[k])
    # u exactly equal to prob[k] rejects (strict <): craft a word with a24 == prob*2^24 in cell 0
    k0 = 0
    t = int(float(prob[k0]) * 2 ** 24)
    if 0 < t < 2 ** 24 and float(prob[k0]) * 2 ** 24 == t:
        w = np.array([(t << 8) // N], np.uint32)   # w*N low word >> 8 == t when N | (t << 8)
        if ((int(w[0]) * N) >> 32) == 0 and (((int(w[0]) * N) & 0xFFFFFFFF) >> 8) == t:
            assert oracle.alias_draw(prob, alias, w)[0] == alias[k0]


def test_draw_matches_python_restatement_of_the_definition(oracle):
    """N equiprobable cells, keep the primary with probability Prob[k] else take Alias[k]."""
    rng = np.random.default_rng(11)
    counts = rng.gamma(0.5, 1.0, 100).astype(np.float32)
    prob, alias = oracle.build_alias(counts)
    words = rng.integers(0, 2 ** 32, 20000, dtype=np.uint64)
    got = oracle.alias_draw(prob, alias, words.astype(np.uint32))
    for w, c in zip(words[:2000], got[:2000]):
        m = int(w) * 100
        k, lo = m >> 32, m & 0xFFFFFFFF
        assert c == (k if (lo >> 8) / 2.0 ** 24 < float(prob[k]) else alias[k])


def test_draw_chi_square_against_source_histogram_and_inverse_cdf(oracle, workloads):
    """north_star: chi-square agreement of alias-sampled frequencies with the source histogram, and with
    a brute-force inverse-CDF sampler fed by the same uniform stream."""
    h = workloads.make_histograms(0, ["iron"], [2.0], 4, 1.0, 300.0, 128, 64, n_draws=200_000)
    rng = np.random.default_rng(5)
    n = 4_000_000
    for counts in (h.counts_dp[0, 1], h.counts_th[0, 2]):
        prob, alias = oracle.build_alias(counts)
        words = rng.integers(0, 2 ** 32, n, dtype=np.uint64).astype(np.uint32)
        cells = oracle.alias_draw(prob, alias, words)
        pmf = counts.astype(np.float64) / counts.sum()
        freq = np.bincount(cells, minlength=len(counts)).astype(np.float64)
        assert np.all(freq[pmf == 0] == 0)
        keep = pmf * n >= 5
        f_obs = np.append(freq[keep], freq[~keep].sum())
        f_exp = np.append(pmf[keep] * n, pmf[~keep].sum() * n)
        sel = f_exp > 0
        assert stats.chisquare(f_obs[sel], f_exp[sel]).pvalue > 0.001
        # brute-force inverse CDF with fresh uniforms: a two-sample chi-square (same distribution)
        cdf = np.cumsum(pmf)
        inv = np.searchsorted(cdf, rng.random(n), side="right").clip(0, len(counts) - 1)
        freq2 = np.bincount(inv, minlength=len(counts)).astype(np.float64)
        both = (freq + freq2) >= 10
        table = np.stack([freq[both], freq2[both]])
        assert stats.chi2_contingency(table)[1] > 0.001
