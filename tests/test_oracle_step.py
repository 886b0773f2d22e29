"""Pins of the oracle's sampling step as a whole: after ONE step at a fixed momentum the
fractional loss and the polar kick of many muons have the closed-form moments of the source histograms (cell pmf
times the log-uniform in-cell law, E[2^t] over a cell = 2^lo (2^d - 1) / (d ln 2)); config 0 ends where the
generator's constants say it must (51 steps, about 48.5 GeV)."""
import numpy as np

from paper_2512_10520_b200.workloads import Geometry, MODE_REGIONS, Muons, REGION_DTYPE


def _cell_moments(counts, axis):
    """mean and variance of v = 2^(lo + (cell + u) d), cell ~ counts, u ~ U[0,1)"""
    pmf = counts.astype(np.float64) / counts.sum()
    lo, d = float(axis[0]), float(axis[1])
    c = np.arange(len(pmf))
    m1 = 2.0 ** (lo + c * d) * (2.0 ** d - 1.0) / (d * np.log(2.0))
    m2 = 4.0 ** (lo + c * d) * (4.0 ** d - 1.0) / (2.0 * d * np.log(2.0))
    mean = (pmf * m1).sum()
    return mean, (pmf * m2).sum() - mean ** 2


def test_one_step_loss_and_scatter_moments(oracle, workloads):
    wl = workloads.config0(n=8, n_draws=200_000)
    T = oracle.OracleTables(wl.hist)
    regs = np.array([(0.0, 1.0, -10.0, 10.0, -10.0, 10.0, 1, 0.0, 0.0, 0.0)], REGION_DTYPE)
    g = Geometry(MODE_REGIONS, -10.0, 10.0, -10.0, 10.0, 0.0, 1.0, 0.5, 1, 0, regions=regs)      # max_steps = 1
    n = 400_000
    for P0, d0 in ((50.0, (0.0, 0.0, 1.0)), (3.7, (0.6, 0.0, 0.8)), (290.0, (0.0, -0.28, 0.96))):
        d0 = np.array(d0)
        pos_q = np.zeros((n, 4), np.float32)
        pos_q[:, 3] = 1.0
        mom = np.zeros((n, 4), np.float32)
        mom[:, :3] = (P0 * d0).astype(np.float32)
        r = oracle.transport(T, g, pos_q, mom, seed=7, threads=oracle.max_threads())
        assert np.all(r["steps"] == 1) and np.all(r["flag"] == 4)
        p1 = r["mom"].astype(np.float64)
        Pin = np.linalg.norm(mom[0, :3].astype(np.float64))
        P1 = np.linalg.norm(p1, axis=1)
        f = 1.0 - P1 / Pin
        theta = np.arccos(np.clip(p1 @ (mom[0, :3].astype(np.float64) / Pin) / P1, -1.0, 1.0))
        i = int(oracle.momentum_bin(T.edges, np.array([Pin], np.float32))[0])
        for name, sample, counts, axis in (("f", f, wl.hist.counts_dp[0, i], wl.hist.axis_dp[0, i]),
                                           ("theta", theta, wl.hist.counts_th[0, i], wl.hist.axis_th[0, i])):
            mean, var = _cell_moments(counts, axis)
            err = abs(sample.mean() - mean)
            assert err < 4.0 * np.sqrt(var / n) + 2e-7 * mean + 1e-9, (P0, name, sample.mean(), mean)
            assert abs(sample.var() - var) < 0.05 * var, (P0, name, sample.var(), var)
        # the kick's azimuth around the incoming direction is uniform: first two Fourier moments vanish
        e1 = np.cross(d0, [0.0, 1.0, 0.0]) if abs(d0[1]) < 0.9 else np.cross(d0, [1.0, 0.0, 0.0])
        e1 /= np.linalg.norm(e1)
        e2 = np.cross(d0, e1)
        phi = np.arctan2(p1 @ e2, p1 @ e1)
        assert abs(np.cos(phi).mean()) < 5.0 / np.sqrt(n) and abs(np.sin(2 * phi).mean()) < 5.0 / np.sqrt(n)
        # straight move of one step length along the post-kick direction (B = 0)
        step = r["pos"].astype(np.float64) - pos_q[:, :3]
        assert np.abs(np.linalg.norm(step, axis=1) - 0.02).max() < 1e-7
        assert np.abs(np.cross(step, p1)).max() < 1e-6 * 0.02 * Pin


def test_config0_ends_where_the_generator_constants_say(oracle, workloads):
    wl = workloads.config0(n=4096, n_draws=200_000)
    r = oracle.transport(oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom), wl.muons.pos_q, wl.muons.mom,
                         wl.seed, threads=oracle.max_threads())
    # 1 m of iron in 2 cm steps: 50 steps inside the slab, the 51st crosses z = 1 m (z advances by < 2 cm per step)
    assert np.all(r["flag"] == 2) and np.all(r["steps"] == 51)
    # Mean loss per step from the generator's constants.  A histogram holds f = Dp/P' for P' ~ U(p_a, p_b) inside its
    # momentum bin, so a muon of momentum P loses on average P * E[Dp(P')/P'] =
    # P * (moyal_mean * ln(p_b/p_a)/(p_b - p_a) + k): Moyal mean = loc + 0.1 loc (gamma + ln 2), loc = 1.5e-3 * 7.874 * 2
    # GeV, and the exponential part Dp = k P' (k = 3e-6 * 7.874 * 2) has f = k whatever P' is.
    loc = 1.5e-3 * 7.874 * 2.0
    moyal_mean = loc * (1.0 + 0.1 * (0.5772156649 + np.log(2.0)))
    k = 3e-6 * 7.874 * 2.0
    edges = 1.0 * 300.0 ** (np.arange(51) / 50.0)
    Pm = 50.0
    for _ in range(51):
        i = np.searchsorted(edges, Pm, side="right") - 1
        pa, pb = edges[i], edges[i + 1]
        Pm -= Pm * (moyal_mean * np.log(pb / pa) / (pb - pa) + k)
    P = np.linalg.norm(r["mom"].astype(np.float64), axis=1)
    assert abs(Pm - 48.5) < 0.1                                      # "about 48.5 GeV"
    assert abs(P.mean() - Pm) < 0.01, (P.mean(), Pm)
    assert np.all(P < 50.0) and np.all(r["pos"][:, 2] >= 1.0) and np.all(r["pos"][:, 2] < 1.02)
