"""Pins for the RK4 Lorentz push (Eq. 4; P-5, P-6, P-7)."""
import math

import numpy as np

# kappa is the float32 constant 0.299792458f in BOTH oracle modes (3e-8 from the exact
# value, 3e-5 from north_star's rounded 0.2998); the closed forms below use the same number.
KAPPA = float(np.float32(0.299792458))
assert abs(KAPPA / 0.299792458 - 1.0) < 4e-8 and abs(KAPPA / 0.2998 - 1.0) < 3e-5


def helix(r0, p0, q, B, s):
    """Closed form for uniform B: p rotates about B by -kappa q |B| s / P; r follows."""
    B = np.asarray(B, float)
    Bn = np.linalg.norm(B)
    P = np.linalg.norm(p0)
    b = B / Bn
    w = KAPPA * q * Bn / P                        # rad per metre of path
    p_par = np.dot(p0, b) * b
    p_perp = p0 - p_par
    c = np.cross(p_perp, b)                       # dp/ds = w (p x b)
    p = p_par + p_perp * math.cos(w * s) + c * math.sin(w * s)
    r = r0 + (p_par * s + p_perp * math.sin(w * s) / w + c * (1 - math.cos(w * s)) / w) / P
    return r, p


def test_straight_line_without_field(oracle):
    r0, p0 = np.array([0.1, -0.2, 0.0]), np.array([1.0, 2.0, 30.0])
    n, h = 500, 0.02
    r, p = oracle.rk4(r0, p0, -1.0, [0, 0, 0], h, n)
    assert np.array_equal(p, p0)
    assert np.abs(r - (r0 + n * h * p0 / np.linalg.norm(p0))).max() < 1e-12
    r32, p32 = oracle.rk4(r0, p0, -1.0, [0, 0, 0], h, n, np.float32)
    assert np.array_equal(p32, p0.astype(np.float32))
    assert np.abs(r32 - (r0 + n * h * p0 / np.linalg.norm(p0))).max() < n * 2.0 ** -23 * 10.0


def test_helix_radius_pitch_and_handedness(oracle):
    # north_star: radius p/(0.2998 q B); F = q v x B: q=+1, p || +z, B || +y bends towards -x
    P, Bmag = 10.0, 1.7
    R = P / (KAPPA * Bmag)
    r, p = oracle.rk4([0, 0, 0], [0, 0, P], +1.0, [0, Bmag, 0], 0.02, 300)
    assert r[0] < 0 and p[0] < 0
    s = 300 * 0.02
    assert abs(r[0] - (-R * (1 - math.cos(s / R)))) < 1e-10
    assert abs(r[2] - R * math.sin(s / R)) < 1e-10
    assert abs(np.linalg.norm(p) - P) < 1e-12 * P
    r, p = oracle.rk4([0, 0, 0], [0, 0, P], -1.0, [0, Bmag, 0], 0.02, 300)
    assert r[0] > 0
    # general direction and field: full closed form, in double and in float32
    r0, p0, B = np.array([0.3, -0.1, 2.0]), np.array([0.7, -0.4, 12.0]), np.array([0.3, 1.7, -0.2])
    for q in (+1.0, -1.0):
        rr, pp = helix(r0, p0, q, B, 400 * 0.02)
        r, p = oracle.rk4(r0, p0, q, B, 0.02, 400)
        assert np.abs(r - rr).max() < 1e-10 and np.abs(p - pp).max() < 1e-9
        r32, p32 = oracle.rk4(r0, p0, q, B, 0.02, 400, np.float32)
        assert np.abs(r32 - rr).max() < 2e-5 and np.abs(p32 - pp).max() < 2e-4
    # momentum parallel to B is untouched
    r, p = oracle.rk4([0, 0, 0], [0, 5.0, 0], 1.0, [0, 1.7, 0], 0.02, 100)
    assert np.array_equal(p, [0, 5.0, 0]) and abs(r[1] - 2.0) < 1e-12


def test_rk4_fourth_order_convergence(oracle):
    # exaggerated curvature so truncation error is visible in double: kappa B h / P ~ 0.2 at h = 2 cm
    P, B, q, L = 0.05, [0.0, 1.7, 0.0], 1.0, 0.32
    r0, p0 = np.zeros(3), np.array([0.01, 0.02, math.sqrt(P * P - 5e-4)])
    rr, pp = helix(r0, p0, q, np.array(B), L)
    errs = []
    for h in (0.02, 0.01, 0.005, 0.0025):
        r, p = oracle.rk4(r0, p0, q, B, h, int(round(L / h)))
        errs.append(max(np.abs(r - rr).max(), np.abs(p - pp).max() / P))
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    # halving h divides the error by 2^4 (from below as h -> 0: the h^5 term has the opposite sign)
    assert all(13.0 < x < 16.5 for x in ratios) and ratios[-1] > 15.0, (errs, ratios)
