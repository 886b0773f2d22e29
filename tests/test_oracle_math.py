"""Pins for the contract's elementary functions and the kick/rotation (P-8)."""
import math

import numpy as np
from scipy import stats

ULP = 2.0 ** -24     # half-unit in the last place of a float32 in [1,2)


def test_exp2c_against_libm(oracle):
    y = np.concatenate([np.linspace(-40, 4, 400001), np.arange(-60, 10), np.arange(-60, 10) + 0.5,
                        np.array([-0.0, 0.0, 1e-20, -1e-20])]).astype(np.float32)
    got = oracle.exp2c(y)
    want = np.exp2(y.astype(np.float64))
    assert (np.abs(got - want) / want).max() < 2.0 * ULP       # <= 2 ulp, like a device exp2f
    assert np.array_equal(oracle.exp2c(np.arange(-100, 100, dtype=np.float32)),
                          np.exp2(np.arange(-100, 100)).astype(np.float32))   # integers are exact
    # clamped outside [-120, 120]
    assert oracle.exp2c(np.array([-500.0], np.float32))[0] == np.float32(2.0 ** -120)
    assert oracle.exp2c(np.array([500.0], np.float32))[0] == np.float32(2.0 ** 120)


def test_sincos_polar_against_libm(oracle):
    th = np.concatenate([np.logspace(-12, math.log10(3.0), 300001), np.linspace(0, 3.0, 100001)]).astype(np.float32)
    s, c = oracle.sincos_polar(th)
    t64 = th.astype(np.float64)
    # sine keeps RELATIVE accuracy for the tiny angles of multiple scattering (theta ~ 1e-6 .. 1e-2)
    m = th > 0
    small = m & (th < 1.5)
    assert (np.abs(s[small] - np.sin(t64[small])) / np.sin(t64[small])).max() < 3.0 * ULP
    assert np.abs(s - np.sin(t64)).max() < 5.0 * ULP
    assert np.abs(c - np.cos(t64)).max() < 5.0 * ULP
    assert oracle.sincos_polar(np.zeros(1, np.float32))[0][0] == 0.0
    assert oracle.sincos_polar(np.zeros(1, np.float32))[1][0] == 1.0
    # angles above pi are clamped to pi
    s, c = oracle.sincos_polar(np.array([10.0], np.float32))
    assert abs(s[0]) < 1e-6 and c[0] == -1.0


def test_sincos_azimuth_against_libm(oracle):
    k = np.concatenate([np.arange(0, 2 ** 24, 5), np.array([0, 2 ** 21 - 1, 2 ** 21, 2 ** 22, 2 ** 23, 3 * 2 ** 22, 2 ** 24 - 1])]).astype(np.uint32)
    s, c = oracle.sincos_azimuth(k)
    phi = 2.0 * math.pi * k.astype(np.float64) / 2 ** 24
    assert np.abs(s - np.sin(phi)).max() < 3.0 * ULP
    assert np.abs(c - np.cos(phi)).max() < 3.0 * ULP
    s, c = oracle.sincos_azimuth(np.array([0, 2 ** 22, 2 ** 23, 3 * 2 ** 22], np.uint32))
    assert np.array_equal(s, np.array([0, 1, 0, -1], np.float32)) and np.array_equal(c, np.array([1, 0, -1, 0], np.float32))


def rodrigues(v, k, theta):
    """PAPER.md Eq. 3 rotation of v about unit axis k by theta."""
    return v * math.cos(theta) + np.cross(k, v) * math.sin(theta) + k * np.dot(k, v) * (1 - math.cos(theta))


def test_frame_is_the_rodrigues_rotation_of_eq3(oracle):
    rng = np.random.default_rng(0)
    for _ in range(500):
        d = rng.standard_normal(3)
        d /= np.linalg.norm(d)
        e1, e2 = oracle.frame(d)
        # orthonormal and right-handed for every direction
        M = np.stack([e1, e2, d])
        assert np.abs(M @ M.T - np.eye(3)).max() < 1e-14
        assert np.abs(np.cross(e1, e2) - d).max() < 1e-14
        if d[2] > 1e-6:
            # Eq. 3: axis k perpendicular to zhat and d, angle between them
            k = np.cross([0, 0, 1.0], d)
            k /= np.linalg.norm(k)
            th = math.acos(d[2])
            assert np.abs(rodrigues(np.array([1.0, 0, 0]), k, th) - e1).max() < 1e-12
            assert np.abs(rodrigues(np.array([0, 1.0, 0]), k, th) - e2).max() < 1e-12
            assert np.abs(rodrigues(np.array([0, 0, 1.0]), k, th) - d).max() < 1e-12
    e1, e2 = oracle.frame(np.array([0, 0, 1.0]))          # Eq. 3 is undefined here; the frame is the identity
    assert np.array_equal(e1, [1, 0, 0]) and np.array_equal(e2, [0, 1, 0])
    e1, e2 = oracle.frame(np.array([0, 0, -1.0]))         # and finite at -z
    assert np.all(np.isfinite(e1)) and np.all(np.isfinite(e2))


def test_kick_geometry(oracle):
    """|p'| = P(1-f); angle to the old direction = theta; azimuth about it = 2 pi k24 / 2^24."""
    rng = np.random.default_rng(1)
    for _ in range(300):
        p = rng.standard_normal(3) * 20.0
        f = 10 ** rng.uniform(-6, -1)
        theta = 10 ** rng.uniform(-5, -0.5)
        k24 = int(rng.integers(0, 2 ** 24))
        P = np.linalg.norm(p)
        d = p / P
        p2, Pn = oracle.kick(p, f, theta, k24)
        assert abs(Pn - P * (1 - f)) < 1e-12 * P
        assert abs(np.linalg.norm(p2) - Pn) < 3e-7 * P           # float32-accurate polynomials
        assert abs(np.dot(p2, d) / Pn - math.cos(theta)) < 3e-7
        e1, e2 = oracle.frame(d)
        phi = math.atan2(np.dot(p2, e2), np.dot(p2, e1)) % (2 * math.pi)
        want = 2 * math.pi * k24 / 2 ** 24
        dphi = (phi - want + math.pi) % (2 * math.pi) - math.pi
        assert abs(dphi) < 1e-5 / max(math.sin(theta), 1e-3) * 1e-2 + 1e-6
    # float32 mode agrees with the double mode
    p = np.array([1.0, -2.0, 30.0])
    a, _ = oracle.kick(p, 1e-3, 2e-3, 12345, np.float32)
    b, _ = oracle.kick(p, 1e-3, 2e-3, 12345, np.float64)
    assert np.abs(a - b).max() < 1e-5


def test_kick_azimuth_is_uniform(oracle):
    rng = np.random.default_rng(4)
    p = np.array([3.0, 4.0, 12.0])
    d = p / np.linalg.norm(p)
    e1, e2 = oracle.frame(d)
    n = 20000
    words = oracle.philox4x32_10(np.stack([np.arange(n), np.zeros(n), np.zeros(n), np.zeros(n)], 1).astype(np.uint32),
                                 np.array([1, 0], np.uint32))
    phis = []
    for w3 in words[:, 3]:
        p2, _ = oracle.kick(p, 1e-3, 1e-2, int(w3 >> 8))
        phis.append(math.atan2(np.dot(p2, e2), np.dot(p2, e1)) % (2 * math.pi))
    hist = np.bincount((np.array(phis) / (2 * math.pi) * 36).astype(int).clip(0, 35), minlength=36)
    assert stats.chisquare(hist).pvalue > 1e-3
