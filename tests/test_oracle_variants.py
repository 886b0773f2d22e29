"""Pins of the oracle's SURVEY.md §8(f) variants (DESIGN.md §3.10 joint 2D histogram mode, §3.11 nearest-neighbour and
per-stage field) against what the paper and the mathematics fix: the exact pmf of an alias table, the geometry of
the kick of PAPER.md L163 / Eq. 3, closed-form cell moments, stored cell values, and the convergence order of RK4."""
import math

import numpy as np
from scipy import stats

from paper_2512_10520_b200.workloads import (FIELD_NEAREST, FIELD_PER_STAGE, Geometry, Histograms, MODE_REGIONS,
                                             MODE_VOXEL, REGION_DTYPE)


# ----------------------------------------------------------------------------------- two-word alias draw
def test_draw2_acceptance_threshold_is_exact(oracle):
    """For a fixed cell k, the number of 24-bit accept values that keep k is ceil(prob[k] 2^24) (u < prob[k] with
    u = a24 2^-24); every other value returns alias[k]."""
    counts = np.array([5.0, 1.0, 0.0, 2.0, 9.0], np.float32)
    prob, alias = oracle.build_alias(counts)
    N = len(counts)
    a24 = np.arange(2 ** 24, dtype=np.uint32)
    for k in range(N):
        w_sel = np.uint32(math.ceil(k * 2 ** 32 / N))             # smallest word with (w N) >> 32 == k
        assert (int(w_sel) * N) >> 32 == k and (k == 0 or ((int(w_sel) - 1) * N) >> 32 == k - 1)
        got = oracle.alias_draw2(prob, alias, np.full(a24.shape, w_sel, np.uint32), a24 << np.uint32(8))
        keep = int((got == k).sum()) if alias[k] != k else None
        if keep is not None:
            assert keep == math.ceil(float(prob[k]) * 2 ** 24)
            assert np.all(got[keep:] == alias[k]) and np.all(got[:keep] == k)
        else:
            assert np.all(got == k)
    # the low 8 bits of the accept word and the select word's low bits never matter; edge words
    w = np.array([0, 0xFFFFFFFF, 0x80000000, 1], np.uint32)
    assert np.array_equal(oracle.alias_draw2(prob, alias, w, np.zeros(4, np.uint32)), [0, 4, 2 if prob[2] > 0 else alias[2], 0])
    assert np.array_equal(oracle.alias_draw2(prob, alias, w, np.full(4, 0xFF, np.uint32)),
                          oracle.alias_draw2(prob, alias, w, np.zeros(4, np.uint32)))


def test_draw2_frequencies_match_the_joint_histogram(oracle, workloads):
    h = workloads.make_histograms(0, ["iron"], [2.0], 3, 1.0, 300.0, 128, 64, n_draws=300_000, joint=True)
    counts = h.counts_dp[0, 1].reshape(-1)
    prob, alias = oracle.build_alias(counts)
    rng = np.random.default_rng(11)
    n = 6_000_000
    ws = rng.integers(0, 2 ** 32, n, dtype=np.uint64).astype(np.uint32)
    wa = rng.integers(0, 2 ** 32, n, dtype=np.uint64).astype(np.uint32)
    cells = oracle.alias_draw2(prob, alias, ws, wa)
    pmf = counts.astype(np.float64) / counts.sum()
    freq = np.bincount(cells, minlength=len(counts)).astype(np.float64)
    assert np.all(freq[pmf == 0] == 0)
    keep = pmf * n >= 5
    f_obs = np.append(freq[keep], freq[~keep].sum())
    f_exp = np.append(pmf[keep] * n, pmf[~keep].sum() * n)
    assert stats.chisquare(f_obs[f_exp > 0], f_exp[f_exp > 0]).pvalue > 0.001
    # brute-force inverse CDF with fresh uniforms: same distribution
    inv = np.searchsorted(np.cumsum(pmf), rng.random(n), side="right").clip(0, len(counts) - 1)
    freq2 = np.bincount(inv, minlength=len(counts)).astype(np.float64)
    both = (freq + freq2) >= 10
    assert stats.chi2_contingency(np.stack([freq[both], freq2[both]]))[1] > 0.001


# ------------------------------------------------------------------------------------------ joint kick
def test_joint_kick_geometry_and_its_reduction_to_the_polar_kick(oracle):
    rng = np.random.default_rng(12)
    for _ in range(300):
        p = rng.standard_normal(3) * rng.uniform(1, 100)
        P = np.linalg.norm(p)
        d = p / P
        fz, ft = 10 ** rng.uniform(-6, -0.5), 10 ** rng.uniform(-7, -1)
        k24 = int(rng.integers(0, 2 ** 24))
        phi = 2 * math.pi * k24 / 2 ** 24
        p1, Pn = oracle.kick_joint(p, fz, ft, k24)
        # dp = [dt cos(phi), dt sin(phi), dz] in the muon's frame with dz = -P fz, dt = P ft
        assert abs(p1 @ d - P * (1 - fz)) < 1e-12 * P
        perp = p1 - (p1 @ d) * d
        assert abs(np.linalg.norm(perp) - P * ft) < 3e-7 * P * ft + 1e-13 * P   # sin^2 + cos^2 of the float32-grade polynomials
        assert abs(Pn - np.linalg.norm(p1)) < 1e-13 * P and abs(Pn - P * math.hypot(1 - fz, ft)) < 1e-9 * P
        e1, e2 = oracle.frame(d)                       # pinned against Eq. 3 in test_oracle_math.py
        assert abs(math.atan2(perp @ e2, perp @ e1) - (phi if phi <= math.pi else phi - 2 * math.pi)) < 1e-6
        # the marginal mode's kick (loss f, polar angle theta) is the joint kick with fz = 1 - (1-f) cos(theta),
        # ft = (1-f) sin(theta): the two must agree (to the float32-grade sin/cos polynomials of the polar kick)
        f, th = 10 ** rng.uniform(-5, -1), 10 ** rng.uniform(-6, -1.5)
        pa, Pa = oracle.kick(p, f, th, k24)
        pb, Pb = oracle.kick_joint(p, 1 - (1 - f) * math.cos(th), (1 - f) * math.sin(th), k24)
        assert np.abs(pa - pb).max() < 3e-7 * P * th + 1e-12 * P and abs(Pa - Pb) < 1e-9 * P
    # float32 mode, start direction exactly +z (config 0) and -z: finite, same geometry
    for pz in (50.0, -50.0):
        p1, Pn = oracle.kick_joint(np.array([0.0, 0.0, pz]), 1e-3, 2e-4, 2 ** 22, np.float32)    # phi = pi/2
        assert np.all(np.isfinite(p1)) and abs(abs(p1[2]) - 50.0 * (1 - 1e-3)) < 1e-5
        assert abs(math.hypot(p1[0], p1[1]) - 50.0 * 2e-4) < 1e-8 and abs(Pn - np.linalg.norm(p1.astype(np.float64))) < 1e-5


def test_joint_one_step_moments_and_decode_order(oracle):
    """After one step the (fz, ft) of many muons have the moments of the 2D table: means of both axes and the mixed
    moment E[fz ft], which a transposed or mis-strided cell decode (n_dp != n_th) would get wrong."""
    # a hand-made, strongly correlated table (large loss <-> large kick), 12 x 5 cells, two momentum bins
    n_a, n_b = 12, 5
    ia, ib = np.meshgrid(np.arange(n_a), np.arange(n_b), indexing="ij")
    counts = np.exp(-((ia / 2.4 - ib) ** 2)).astype(np.float32)
    counts[3, 4] = 0.0
    hist = Histograms(1, 2, n_a, n_b, 1.0, 300.0, np.stack([counts, counts[::-1].copy()])[None], None,
                      np.zeros((1, 2, 2), np.float32) + [-11.0, 0.45], np.zeros((1, 2, 2), np.float32) + [-13.0, 1.1],
                      np.array([0.02, 0.02], np.float32), joint=True)
    T = oracle.OracleTables(hist)
    regs = np.array([(0.0, 1.0, -10.0, 10.0, -10.0, 10.0, 1, 0.0, 0.0, 0.0)], REGION_DTYPE)
    g = Geometry(MODE_REGIONS, -10.0, 10.0, -10.0, 10.0, 0.0, 1.0, 0.5, 1, 0, regions=regs)
    n = 500_000
    pos_q = np.zeros((n, 4), np.float32)
    pos_q[:, 3] = -1.0
    mom = np.zeros((n, 4), np.float32)
    mom[:, :3] = np.array([3.0, -4.0, 12.0], np.float32)                       # |p| = 13
    r = oracle.transport(T, g, pos_q, mom, seed=3, threads=oracle.max_threads())
    assert np.all(r["steps"] == 1)
    p1 = r["mom"].astype(np.float64)
    d = np.array([3.0, -4.0, 12.0]) / 13.0
    fz = 1.0 - (p1 @ d) / 13.0
    ft = np.linalg.norm(p1 - np.outer(p1 @ d, d), axis=1) / 13.0
    i = int(oracle.momentum_bin(T.edges, np.array([13.0], np.float32))[0])
    assert i == 0
    pmf = counts.astype(np.float64) / counts.sum()

    def cell_mean(axis, ncell):
        lo, dd = float(axis[0]), float(axis[1])
        return 2.0 ** (lo + np.arange(ncell) * dd) * (2.0 ** dd - 1.0) / (dd * math.log(2.0))
    ma, mb = cell_mean(hist.axis_dp[0, i], n_a), cell_mean(hist.axis_th[0, i], n_b)
    Ea, Eb, Eab = (pmf.sum(1) * ma).sum(), (pmf.sum(0) * mb).sum(), (pmf * np.outer(ma, mb)).sum()
    assert abs(fz.mean() - Ea) < 5 * fz.std() / math.sqrt(n) + 1e-6 * Ea
    assert abs(ft.mean() - Eb) < 5 * ft.std() / math.sqrt(n) + 1e-6 * Eb
    assert abs((fz * ft).mean() - Eab) < 5 * (fz * ft).std() / math.sqrt(n) + 1e-6 * Eab
    assert abs(Eab - Ea * Eb) > 20 * (fz * ft).std() / math.sqrt(n)            # the table IS correlated: the check bites


# ------------------------------------------------------------------------------------- field variants
def _vacuum_tables(h):
    return Histograms(1, 2, 4, 4, 1.0, 300.0, np.ones((1, 2, 4), np.float32), np.ones((1, 2, 4), np.float32),
                      np.zeros((1, 2, 2), np.float32) + [-10.0, 0.1], np.zeros((1, 2, 2), np.float32) + [-10.0, 0.1],
                      np.array([h, 0.01], np.float32))


def test_nearest_field_is_the_stored_cell_value(oracle):
    rng = np.random.default_rng(13)
    nx, ny, nz, cell = 9, 6, 11, 0.125
    fld = rng.standard_normal((nz, ny, nx, 3)).astype(np.float32)
    mat = rng.integers(0, 3, (nz, ny, nx)).astype(np.uint8)
    g = Geometry(MODE_VOXEL, -9.0, 9.0, -9.0, 9.0, -9.0, 9.0, 1.0, 10, 2, nx=nx, ny=ny, nz=nz, ox=-0.5, oy=0.25, oz=1.0,
                 cell=cell, material=mat, field=fld, field_mode=FIELD_NEAREST)
    pts = (np.array([-0.5, 0.25, 1.0]) + rng.random((20000, 3)) * np.array([nx, ny, nz]) * cell).astype(np.float32)
    idx = np.floor((pts - np.array([-0.5, 0.25, 1.0], np.float32)) * np.float32(8.0)).astype(int)
    m, B = oracle.material_and_field(g, pts, dtype=np.float32)
    assert np.array_equal(B, fld[idx[:, 2], idx[:, 1], idx[:, 0]]) and np.array_equal(m, mat[idx[:, 2], idx[:, 1], idx[:, 0]])
    out = np.array([[-0.6, 0.5, 1.5], [0.0, 0.5, 1.0 + nz * cell]], np.float32)
    m, B = oracle.material_and_field(g, out, dtype=np.float32)
    assert np.all(B == 0) and np.all(m == 2)
    # at cell centres nearest and trilinear agree (both return the stored value)
    g.field_mode = 0
    ctr = (np.array([-0.5, 0.25, 1.0]) + (idx[:500] + 0.5) * cell).astype(np.float32)
    _, Bt = oracle.material_and_field(g, ctr, dtype=np.float32)
    assert np.array_equal(Bt, fld[idx[:500, 2], idx[:500, 1], idx[:500, 0]])


def _gradient_geometry(field_mode, h, n_steps):
    # vacuum everywhere (no sampling); By = 1.7 + 1.2 x [T] on a 5-cm grid: trilinear reproduces it exactly
    nx, ny, nz, cell = 48, 8, 64, 0.05
    xc = -1.2 + (np.arange(nx) + 0.5) * cell
    fld = np.zeros((nz, ny, nx, 3), np.float32)
    fld[..., 1] = (1.7 + 1.2 * xc).astype(np.float32)[None, None, :]
    mat = np.zeros((nz, ny, nx), np.uint8)
    return Geometry(MODE_VOXEL, -1.2, 1.2, -0.2, 0.2, 0.0, 3.2, 0.01, n_steps, 0, nx=nx, ny=ny, nz=nz, ox=-1.2, oy=-0.2,
                    oz=0.0, cell=cell, material=mat, field=fld, field_mode=field_mode)


def _push(oracle, field_mode, h, length=1.6):
    n = int(round(length / h))
    g = _gradient_geometry(field_mode, h, n)
    T = oracle.OracleTables(_vacuum_tables(h))
    pos_q = np.array([[0.05, 0.01, 0.3, 1.0]])
    mom = np.array([[0.05, 0.02, 0.45, 0.0]])
    r = oracle.transport(T, g, pos_q, mom, seed=1, dtype=np.float64)
    assert r["flag"][0] == 4 and r["steps"][0] == n
    return np.concatenate([r["pos"][0], r["mom"][0]])


def test_per_stage_push_is_fourth_order_in_a_field_gradient_and_frozen_is_first_order(oracle):
    ref = _push(oracle, FIELD_PER_STAGE, 0.003125)
    err_stage = [np.abs(_push(oracle, FIELD_PER_STAGE, h) - ref)[:3].max() for h in (0.1, 0.05, 0.025)]
    err_frozen = [np.abs(_push(oracle, 0, h) - ref)[:3].max() for h in (0.1, 0.05, 0.025)]
    assert 12.0 < err_stage[0] / err_stage[1] < 20.0 and 12.0 < err_stage[1] / err_stage[2] < 20.0      # h^4
    assert 1.7 < err_frozen[0] / err_frozen[1] < 2.4 and 1.7 < err_frozen[1] / err_frozen[2] < 2.4    # h^1 (R-7)
    assert err_stage[2] < 1e-3 * err_frozen[2]
    # |p| is conserved by the exact flow; RK4 keeps it to O(h^4) per unit length
    assert abs(np.linalg.norm(_push(oracle, FIELD_PER_STAGE, 0.025)[3:]) - np.linalg.norm([0.05, 0.02, 0.45])) < 1e-7


def test_per_stage_equals_frozen_in_a_uniform_field_and_sees_region_boundaries(oracle, workloads):
    # one magnetised region: every stage sees the same B, so the two pushes are the same float32 operations
    wl = workloads.config1(n=3000, n_draws=20_000)
    T = oracle.OracleTables(wl.hist)
    wl.geom.max_steps = 40
    a = oracle.transport(T, oracle.OracleGeometry(wl.geom), wl.muons.pos_q, wl.muons.mom, 1, threads=4)
    wl.geom.field_mode = FIELD_PER_STAGE
    b = oracle.transport(T, oracle.OracleGeometry(wl.geom), wl.muons.pos_q, wl.muons.mom, 1, threads=4)
    inside = np.all(np.abs(a["pos"][:, :2]) < 0.9, axis=1) & (a["flag"] == 4)
    assert inside.sum() > 2000
    for k in ("pos", "mom"):
        assert np.array_equal(a[k][inside], b[k][inside])
    # vacuum, field only for z >= 1: a 10-cm step starting at z = 0.95 is straight when frozen, bent per stage
    regs = np.array([(1.0, 2.0, -5.0, 5.0, -5.0, 5.0, 0, 0.0, 1.7, 0.0)], REGION_DTYPE)
    g = Geometry(MODE_REGIONS, -5.0, 5.0, -5.0, 5.0, 0.0, 9.0, 0.01, 1, 0, regions=regs)
    Tv = oracle.OracleTables(_vacuum_tables(0.1))
    pos_q, mom = np.array([[0.0, 0.0, 0.95, 1.0]]), np.array([[0.0, 0.0, 1.0, 0.0]])
    fr = oracle.transport(Tv, g, pos_q, mom, 1, dtype=np.float64)
    assert np.array_equal(fr["mom"][0], [0.0, 0.0, 1.0]) and abs(fr["pos"][0][2] - 1.05) < 1e-8   # h and h/6 are float32 constants
    g.field_mode = FIELD_PER_STAGE
    st = oracle.transport(Tv, g, pos_q, mom, 1, dtype=np.float64)
    # stages 2 and 3 sit at z = 1.0 (inside), stage 4 at 1.05: dpx = -(h/6) kappa B (0 + 2 + 2 + 1) to first order
    kappa = float(np.float32(0.299792458))
    assert abs(st["mom"][0][0] + 0.1 / 6 * kappa * 1.7 * 5) < 2e-3 and st["mom"][0][0] < 0
