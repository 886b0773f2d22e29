"""Pins for log momentum binning (P-4)."""
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_momentum_bins.txt")


def test_edges_reproduce_the_papers_worked_example(oracle):
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    n, lo, hi, b_lo, b_hi, dec = rows[0]
    n, dec = int(n), int(dec)
    e = oracle.make_edges(float(lo), float(hi), n)
    assert len(e) == n + 1 and e.dtype == np.float32
    # exactly one bin rounds to the printed pair; "95 bins" are 95 intervals
    hits = [j for j in range(n) if round(float(e[j]), dec) == float(b_lo) and round(float(e[j + 1]), dec) == float(b_hi)]
    assert hits == [80]
    assert e[0] == np.float32(float(lo)) and abs(float(e[-1]) - float(hi)) < 1e-4
    assert np.all(np.diff(e) > 0)
    assert np.allclose(e[1:] / e[:-1], (float(hi) / float(lo)) ** (1.0 / n), rtol=1e-6)


def test_momentum_bin_equals_linear_scan(oracle):
    e = oracle.make_edges(1.0, 300.0, 50)
    rng = np.random.default_rng(2)
    P = np.concatenate([np.exp(rng.uniform(np.log(0.5), np.log(400.0), 20000)).astype(np.float32),
                        e, np.nextafter(e, np.float32(0)), np.nextafter(e, np.float32(1e9)),
                        np.array([0.0, 1e-30, 1e30, np.inf], np.float32)])
    got = oracle.momentum_bin(e, P)
    for p, g in zip(P, got):
        want = 0
        for j in range(50):                       # brute force: last j with e[j] <= P, clamped
            if e[j] <= p:
                want = j
        assert g == want
