"""Pin of the oracle's break-test block (oracle/muon_oracle.cpp, top of transport_one): Algorithm 1 l.2-4
 as read in DESIGN.md §3.1 / R-2 —

    !(P >= p_min) -> STOPPED (1);  z >= z_exit -> EXITED (2);
    x < x_min || x >= x_max || y < y_min || y >= y_max || z < z_min -> ESCAPED (3);  step == max_steps -> MAXSTEPS (4)

tested in that order.  Every expectation below is a literal worked out by hand from that text, on a world of vacuum
(no sampling, no field: a muon that passes the tests moves h = 0.25 m along its momentum and is tested again), so a
wrong comparison (`x > x_max`, `P > p_min`), a missing side of the box, a NaN that slips through, or a swapped priority
fails here on the CPU, in float32 and in float64 mode.
"""
import numpy as np
import pytest

from paper_2512_10520_b200.workloads import Geometry, Histograms, MODE_REGIONS

STOPPED, EXITED, ESCAPED, MAXSTEPS = 1, 2, 3, 4
H = 0.25          # step length in vacuum (an exact binary fraction: positions stay exact)


def _tables(oracle):
    """one material that is never entered; step_m[0] = H is the vacuum step"""
    one = np.ones((1, 1, 4), np.float32)
    ax = np.array([[[-10.0, 0.5]]], np.float32)
    h = Histograms(1, 1, 4, 4, 1.0, 300.0, one, one.copy(), ax, ax.copy(), np.array([H, H], np.float32))
    return oracle.OracleTables(h)


def _world(max_steps):
    # world box x in [-1, 1), y in [-2, 3), z in [0.5, 2), all vacuum; p_min = 1.5
    return Geometry(MODE_REGIONS, -1.0, 1.0, -2.0, 3.0, 0.5, 2.0, 1.5, max_steps, 0, regions=None)


def _run(oracle, dtype, max_steps, pos, mom):
    pos_q = np.zeros((1, 4), dtype)
    pos_q[0, :3], pos_q[0, 3] = pos, 1.0
    m = np.zeros((1, 4), dtype)
    m[0, :3] = mom
    r = oracle.transport(_tables(oracle), _world(max_steps), pos_q, m, seed=3, dtype=dtype)
    return int(r["flag"][0]), int(r["steps"][0]), r["pos"][0], r["mom"][0]


def _below(v, dtype):
    return np.nextafter(dtype(v), dtype(-np.inf))


def _above(v, dtype):
    return np.nextafter(dtype(v), dtype(np.inf))


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_momentum_cut(oracle, dtype):
    mid = (0.0, 0.0, 1.0)
    # P one ulp below p_min -> STOPPED at once; P == p_min passes (the test is P >= p_min); zero and NaN stop
    assert _run(oracle, dtype, 5, mid, (0, 0, _below(1.5, dtype)))[:2] == (STOPPED, 0)
    assert _run(oracle, dtype, 1, mid, (0, 0, 1.5))[:2] == (MAXSTEPS, 1)
    assert _run(oracle, dtype, 5, mid, (0, 0, 0))[:2] == (STOPPED, 0)
    assert _run(oracle, dtype, 5, mid, (np.nan, 0, 5))[:2] == (STOPPED, 0)
    assert _run(oracle, dtype, 5, mid, (0, 0, -np.nan))[:2] == (STOPPED, 0)
    # |p| is the norm of all three components: (0.9, 1.2, 0) has P = 1.5 exactly (passes), (0.9, 1.1, 0) does not
    assert _run(oracle, dtype, 1, mid, (0.9, 1.2, 0))[:2] == (MAXSTEPS, 1)
    assert _run(oracle, dtype, 5, mid, (0.9, 1.1, 0))[:2] == (STOPPED, 0)
    # a stopped muon keeps the state it had at the break
    f, s, pos, mom = _run(oracle, dtype, 5, (0.25, -0.5, 1.0), (0.5, 0.25, 1.0))
    assert (f, s) == (STOPPED, 0) and np.array_equal(pos, dtype([0.25, -0.5, 1.0])) and np.array_equal(mom, dtype([0.5, 0.25, 1.0]))


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_exit_plane(oracle, dtype):
    up = (0, 0, 4.0)
    # z exactly on the plane -> EXITED without a step; one ulp below it -> one step of H, then EXITED at z = 2 - ulp + H
    assert _run(oracle, dtype, 5, (0, 0, 2.0), up)[:2] == (EXITED, 0)
    f, s, pos, _ = _run(oracle, dtype, 5, (0, 0, _below(2.0, dtype)), up)
    assert (f, s) == (EXITED, 1) and 2.0 < float(pos[2]) < 2.2500001
    # from z = 1: steps end at 1.25, 1.5, 1.75, 2.0 -> the 4th reaches the plane (>=, not >).  Exact in float32 (the
    # contract's h/6 is a float32 constant, so float64 mode moves 0.25 (1 + 6e-8) per step: it lands just behind the plane)
    f, s, pos, _ = _run(oracle, dtype, 50, (0, 0, 1.0), up)
    assert (f, s) == (EXITED, 4) and (pos[2] == 2.0 if dtype == np.float32 else abs(pos[2] - 2.0) < 1e-6)
    # beyond the plane is still EXITED (not ESCAPED), whatever x and y are inside the box
    assert _run(oracle, dtype, 5, (0.5, 2.5, 7.0), up)[:2] == (EXITED, 0)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_world_box_is_half_open_on_both_sides(oracle, dtype):
    up = (0, 0, 4.0)            # moves along z only: x and y keep their start values
    inside = (MAXSTEPS, 1)      # passes the tests at step 0, takes the one allowed step
    out = (ESCAPED, 0)
    assert _run(oracle, dtype, 1, (-1.0, 0, 1.0), up)[:2] == inside            # x == x_min is inside
    assert _run(oracle, dtype, 1, (_below(-1.0, dtype), 0, 1.0), up)[:2] == out
    assert _run(oracle, dtype, 1, (1.0, 0, 1.0), up)[:2] == out                # x == x_max is outside
    assert _run(oracle, dtype, 1, (_below(1.0, dtype), 0, 1.0), up)[:2] == inside
    assert _run(oracle, dtype, 1, (0, -2.0, 1.0), up)[:2] == inside            # y == y_min is inside
    assert _run(oracle, dtype, 1, (0, _below(-2.0, dtype), 1.0), up)[:2] == out
    assert _run(oracle, dtype, 1, (0, 3.0, 1.0), up)[:2] == out                # y == y_max is outside
    assert _run(oracle, dtype, 1, (0, _below(3.0, dtype), 1.0), up)[:2] == inside
    assert _run(oracle, dtype, 1, (0, 0, 0.5), up)[:2] == inside               # z == z_min is inside
    assert _run(oracle, dtype, 1, (0, 0, _below(0.5, dtype)), up)[:2] == out   # z < z_min: backwards out
    # x and y are tested against their OWN bounds (a swapped pair would pass these: |x| < 1 but y in [-2, 3))
    assert _run(oracle, dtype, 1, (0, 2.5, 1.0), up)[:2] == inside
    assert _run(oracle, dtype, 1, (0, -1.5, 1.0), up)[:2] == inside
    assert _run(oracle, dtype, 1, (2.5, 0, 1.0), up)[:2] == out
    assert _run(oracle, dtype, 1, (-1.5, 0, 1.0), up)[:2] == out
    # NaN position: every comparison is false -> not exited, not escaped -> runs into the step cap
    assert _run(oracle, dtype, 1, (np.nan, 0, 1.0), up)[:2] == (MAXSTEPS, 1)
    # a muon walking sideways leaves through x_max = 1: from x = 0 with H = 0.25 it is at 1.0 after 4 steps
    f, s, pos, _ = _run(oracle, dtype, 50, (0, 0, 1.0), (4.0, 0, 0))
    assert (f, s) == (ESCAPED, 4) and (pos[0] == 1.0 if dtype == np.float32 else abs(pos[0] - 1.0) < 1e-6)
    # and through x_min = -1 only one step later: x = -1.0 after 4 steps is still inside (float32, where the steps are
    # exact; float64 mode is 6e-8 beyond it by then, see test_exit_plane)
    f, s, pos, _ = _run(oracle, dtype, 50, (0, 0, 1.0), (-4.0, 0, 0))
    assert (f, s, float(pos[0])) == (ESCAPED, 5, -1.25) if dtype == np.float32 else (f, s) == (ESCAPED, 4)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_step_cap(oracle, dtype):
    up = (0, 0, 4.0)
    assert _run(oracle, dtype, 0, (0, 0, 1.0), up)[:2] == (MAXSTEPS, 0)
    f, s, pos, _ = _run(oracle, dtype, 3, (0, 0, 1.0), up)
    assert (f, s) == (MAXSTEPS, 3) and (pos[2] == 1.75 if dtype == np.float32 else abs(pos[2] - 1.75) < 1e-6)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_priority_order(oracle, dtype):
    """STOPPED > EXITED > ESCAPED > MAXSTEPS when several conditions hold at once (max_steps = 0 makes the last one
    hold for every muon here)."""
    slow, fast = (0, 0, 1.0), (0, 0, 4.0)            # below / above the cut p_min = 1.5
    past, before = 2.5, 1.0                          # behind / in front of the exit plane z = 2
    outside, inside = 1.5, 0.0                       # x outside / inside the box
    assert _run(oracle, dtype, 0, (outside, 0, past), slow)[:2] == (STOPPED, 0)      # all four hold
    assert _run(oracle, dtype, 0, (inside, 0, past), slow)[:2] == (STOPPED, 0)       # cut + plane + cap
    assert _run(oracle, dtype, 0, (outside, 0, before), slow)[:2] == (STOPPED, 0)    # cut + box + cap
    assert _run(oracle, dtype, 0, (inside, 0, before), slow)[:2] == (STOPPED, 0)     # cut + cap
    assert _run(oracle, dtype, 0, (outside, 0, past), fast)[:2] == (EXITED, 0)       # plane + box + cap
    assert _run(oracle, dtype, 0, (inside, 0, past), fast)[:2] == (EXITED, 0)        # plane + cap
    assert _run(oracle, dtype, 0, (outside, 0, before), fast)[:2] == (ESCAPED, 0)    # box + cap
    assert _run(oracle, dtype, 0, (inside, 0, before), fast)[:2] == (MAXSTEPS, 0)    # cap only
    # the same with the cap not reached: the first three keep their order
    assert _run(oracle, dtype, 9, (outside, 0, past), slow)[:2] == (STOPPED, 0)
    assert _run(oracle, dtype, 9, (outside, 0, past), fast)[:2] == (EXITED, 0)
    assert _run(oracle, dtype, 9, (outside, 0, before), fast)[:2] == (ESCAPED, 0)
    # z below z_min together with a y outside: still ESCAPED; z below z_min with a momentum below the cut: STOPPED
    assert _run(oracle, dtype, 9, (0, 5.0, 0.25), fast)[:2] == (ESCAPED, 0)
    assert _run(oracle, dtype, 9, (0, 0, 0.25), slow)[:2] == (STOPPED, 0)
    # conditions that start to hold together after a step: from (0.75, 0, 1.75) along (+x, +z) one step of H ends at
    # x = 0.75 + H/sqrt(2) < 1 ... use an axis-aligned case instead: diagonal in x and z with |p| = 5 = (3, 0, 4):
    # dx = 0.15, dz = 0.2 per step; from (0.85, 0, 1.8): after one step x = 1.0 (outside) and z = 2.0 (on the plane) in
    # exact arithmetic; both modes must call it EXITED or — if rounding leaves z a hair below 2 — ESCAPED, never MAXSTEPS
    f, s, pos, _ = _run(oracle, np.float64, 9, (0.85, 0, 1.8), (3.0, 0, 4.0))
    assert s == 1 and f == (EXITED if pos[2] >= 2.0 else ESCAPED)
