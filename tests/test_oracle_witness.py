"""The libm witness (oracle `libm=True`; R-21, §9): Algorithm 1 with the C library's exp2 / sin / cos in
place of the fixed polynomials of DESIGN.md §3.6 and the azimuth written as phi = 2 pi u.  The
contract-mode oracle must agree with it at north_star's REAL tolerance — at least 99.9 % of muons with the same flag
and step count, |dP|/P <= 1e-5 and |dr| <= 1e-5 m — and the two final-state populations must pass the two-sample
KS test (p > 0.01) on p, theta, x, y.  This pins the polynomials inside the whole loop against the plain
definitions: a wrong coefficient, a swapped sin/cos, a wrong quadrant or a jitter decoded on the wrong axis moves
every muon by far more than 1e-5.  (The -m gpu twin, tests/test_gpu_witness.py, holds the CUDA path to the same.)
"""
import numpy as np

from gpu_util import compare, ks_populations

MATCH = 0.999


def _both(oracle, wl):
    T, G = oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom)
    th = oracle.max_threads()
    a = oracle.transport(T, G, wl.muons.pos_q, wl.muons.mom, wl.seed, threads=th)
    b = oracle.transport(T, G, wl.muons.pos_q, wl.muons.mom, wl.seed, threads=th, libm=True)
    return a, b


def check_against_witness(got, witness, label):
    """north_star's criteria; returns the comparison for reporting"""
    c = compare(got, witness)
    ks = ks_populations(got, witness)
    residual = ~c["mask"]
    print("[witness] %s: matched %.5f (bit-exact %.3f), residual %d, max |dP|/P %.2e, max |dr| %.2e, KS %s"
          % (label, c["matched"], c["bit_exact"], residual.sum(), c["max_dp"], c["max_dr"],
             {k: round(float(v), 3) for k, v in ks.items()}))
    assert c["matched"] >= MATCH, (label, c["matched"])
    assert min(ks.values()) > 0.01, (label, ks)
    if residual.sum() >= 100:            # the residual subset on its own when it is large enough
        sub = lambda d: {k: d[k][residual] for k in ("pos", "mom")}
        ks_res = ks_populations(sub(got), sub(witness))
        print("[witness] %s: KS on the %d residual muons alone %s" % (label, residual.sum(), {k: round(float(v), 3) for k, v in ks_res.items()}))
        assert min(ks_res.values()) > 0.01, (label, ks_res)
    # the witness is NOT the contract: if every muon were bit-identical the two modes would be the same code
    assert c["bit_exact"] < 1.0
    return c


def test_config1_contract_matches_libm_witness(oracle, workloads):
    wl = workloads.config1(n=32768, n_draws=60_000)
    a, b = _both(oracle, wl)
    check_against_witness(a, b, "config1 (32768 muons)")


def test_config3_small_contract_matches_libm_witness(oracle, workloads):
    wl = workloads.config3(n=20_000, n_draws=40_000, n_cells=2, half_width_cells=40)
    a, b = _both(oracle, wl)
    check_against_witness(a, b, "config3 small (20000 muons, 80x80x750 grid)")


def test_joint_mode_contract_matches_libm_witness(oracle, workloads):
    """The same bar for the paper's joint 2D tables: there exp2c decodes BOTH sampled
    values (the longitudinal loss fz and the transverse kick ft, which replaces the polar angle and its sine / cosine) and
    the new |p| comes from one more square root — none of which the marginal-mode witness runs exercise."""
    wl = workloads.config1(n=32768, n_draws=100_000, joint=True)
    a, b = _both(oracle, wl)
    check_against_witness(a, b, "config1 joint (32768 muons)")
    wl = workloads.config3(n=20_000, n_draws=40_000, n_cells=2, half_width_cells=40, joint=True, table_shape=(100, 64, 32))
    a, b = _both(oracle, wl)
    check_against_witness(a, b, "config3 small joint (20000 muons, 80x80x750 grid)")


def test_witness_in_double_is_the_physics_mode(oracle, workloads):
    """In float64 the polynomials (float32-accurate, ~1e-7) and libm differ at the 1e-7 level per sampled value, so the
    two double-precision runs agree on flag and step count for nearly every muon and on |p| to ~1e-6 relative:
    the polynomials are accurate to float32 and no better, which is all the contract claims (R-21)."""
    wl = workloads.config1(n=4096, n_draws=60_000)
    T, G = oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom)
    a = oracle.transport(T, G, wl.muons.pos_q, wl.muons.mom, wl.seed, dtype=np.float64, threads=oracle.max_threads())
    b = oracle.transport(T, G, wl.muons.pos_q, wl.muons.mom, wl.seed, dtype=np.float64, threads=oracle.max_threads(), libm=True)
    same = (a["flag"] == b["flag"]) & (a["steps"] == b["steps"])
    assert same.mean() >= 0.999
    Pa, Pb = np.linalg.norm(a["mom"], axis=1), np.linalg.norm(b["mom"], axis=1)
    rel = np.abs(Pa - Pb)[same] / Pb[same]
    assert 1e-12 < np.median(rel) < 1e-5 and np.quantile(rel, 0.99) < 1e-4
