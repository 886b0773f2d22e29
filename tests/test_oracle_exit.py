"""Pins of the oracle's exit-plane projection against closed forms: the exact plane
crossing of a straight line, and the sagitta of a circular arc in a uniform field (error quadratic in the overshoot)."""
import numpy as np

from paper_2512_10520_b200.workloads import Geometry, Histograms, MODE_REGIONS, REGION_DTYPE

KAPPA = 0.299792458


def test_straight_lines_are_recovered_exactly(oracle):
    # vacuum world, no field: the track is r0 + s d; Algorithm 1 stops it up to one step behind the plane, the projection
    # must put it back at r0 + d (z_exit - z0) / dz
    rng = np.random.default_rng(31)
    n = 2000
    one = np.ones((1, 2, 4), np.float32)
    ax = np.zeros((1, 2, 2), np.float32) + [-10.0, 0.5]
    hist = Histograms(1, 2, 4, 4, 1.0, 300.0, one, one.copy(), ax, ax.copy(), np.array([0.07, 0.02], np.float32))
    geom = Geometry(MODE_REGIONS, -50.0, 50.0, -50.0, 50.0, -1.0, 3.0, 0.5, 100000, 0, regions=np.zeros(0, REGION_DTYPE))
    d = rng.standard_normal((n, 3)); d[:, 2] = np.abs(d[:, 2]) + 0.3
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    P = rng.uniform(2.0, 100.0, n)
    pos_q = np.c_[rng.uniform(-1, 1, (n, 2)), rng.uniform(-0.5, 0.5, n), np.where(np.arange(n) % 2, 1.0, -1.0)]
    mom = np.c_[d * P[:, None], np.zeros(n)]
    out = oracle.transport(oracle.OracleTables(hist), oracle.OracleGeometry(geom), pos_q, mom, 1, dtype=np.float64)
    assert np.all(out["flag"] == 2)
    over = out["pos"][:, 2] - 3.0
    assert np.all(over >= 0) and np.all(over < 0.07) and over.max() > 0.03            # the break overshoots
    got = oracle.exit_project(out["pos"], out["mom"], 3.0, dtype=np.float64)
    want = pos_q[:, :3] + d * ((3.0 - pos_q[:, 2]) / d[:, 2])[:, None]
    assert np.all(got[:, 2] == 3.0)
    assert np.abs(got - want).max() < 1e-11
    # float32: the same to rounding of the 3 m lever arm
    got32 = oracle.exit_project(out["pos"].astype(np.float32), out["mom"].astype(np.float32), 3.0, dtype=np.float32)
    assert got32.dtype == np.float32 and np.abs(got32 - want).max() < 5e-6


def test_sagitta_in_a_uniform_field_and_untouched_cases(oracle):
    # circle of radius R = P / (kappa B) in the xz-plane (B along y): a point an arc length L behind the plane, projected
    # back along its tangent, misses the true crossing by the sagitta L^2 / (2R) to first order — quadratic in the overshoot
    P, B = 10.0, 1.7
    R = P / (KAPPA * B)
    errs = []
    for L in (0.04, 0.02, 0.01):
        phi = L / R                                            # crossing at angle 0: x = R, z = 0, tangent +z
        pos = np.array([[R * np.cos(phi), 0.3, R * np.sin(phi)]])
        mom = np.array([[-P * np.sin(phi), 0.0, P * np.cos(phi)]])
        got = oracle.exit_project(pos, mom, 0.0, dtype=np.float64)
        assert got[0, 2] == 0.0 and got[0, 1] == 0.3
        errs.append(got[0, 0] - R)
    want = [L * L / (2 * R) for L in (0.04, 0.02, 0.01)]
    assert np.allclose(errs, want, rtol=1e-3)                  # 4.1e-5 m at a 4 cm overshoot, 2.5e-6 at 1 cm
    assert abs(errs[0] / errs[1] - 4.0) < 0.01 and abs(errs[1] / errs[2] - 4.0) < 0.01
    # pz <= 0 or NaN: left alone; the momentum is never touched (it is an input only)
    pos = np.array([[1.0, 2.0, 3.5], [1.0, 2.0, 3.5], [1.0, 2.0, 3.5]])
    mom = np.array([[1.0, 1.0, 0.0], [1.0, 1.0, -2.0], [1.0, 1.0, np.nan]])
    assert np.array_equal(oracle.exit_project(pos, mom, 3.0, dtype=np.float64), pos)
    assert np.array_equal(oracle.exit_project(pos.astype(np.float32), mom.astype(np.float32), 3.0), pos.astype(np.float32))
