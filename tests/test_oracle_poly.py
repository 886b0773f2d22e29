"""Pins of the oracle's convex-polyhedra lookup (§4.1, Eq. 2) against things other
than itself: scipy's convex hull of a block's eight vertices (an independent library routine), the closed-form
volume of a prismatoid, the axis-aligned boxes of the regions lookup, and the symmetries the test must have."""
import numpy as np
import pytest
from scipy.spatial import ConvexHull

from paper_2512_10520_b200 import workloads as w
from paper_2512_10520_b200.workloads import Geometry, MODE_POLY, MODE_REGIONS, POLY_DTYPE

WORLD = 3


def _geom(blocks, **kw):
    return Geometry(MODE_POLY, -100.0, 100.0, -100.0, 100.0, -100.0, 100.0, 1.0, 10, WORLD,
                    blocks=np.asarray(blocks, POLY_DTYPE), **kw)


def _block(z_lo, z_hi, lo, hi, material=1, B=(0.0, 0.0, 0.0)):
    b = np.zeros((), POLY_DTYPE)
    b["z_lo"], b["z_hi"], b["xy_lo"], b["xy_hi"], b["material"] = z_lo, z_hi, lo, hi, material
    b["bx"], b["by"], b["bz"] = B
    return b


def _convex_quad(rng, centre, radius):
    # four points on an ellipse at increasing angles: convex, counter-clockwise
    ang = np.sort(rng.uniform(0, 2 * np.pi, 4))
    while np.min(np.diff(np.concatenate([ang, [ang[0] + 2 * np.pi]]))) < 0.5:
        ang = np.sort(rng.uniform(0, 2 * np.pi, 4))
    return np.stack([centre[0] + radius[0] * np.cos(ang), centre[1] + radius[1] * np.sin(ang)], -1)


def _frustum(rng):
    """A block whose side faces are planar: the upper face is the lower one scaled and shifted, so the solid is the
    convex hull of its eight vertices and the interpolated slice is the hull's true cross-section."""
    lo = _convex_quad(rng, rng.uniform(-1, 1, 2), rng.uniform(0.5, 2.0, 2))
    s, shift = rng.uniform(0.3, 1.7), rng.uniform(-1, 1, 2)
    hi = lo * s + shift
    z_lo = rng.uniform(-3, 3)
    return _block(z_lo, z_lo + rng.uniform(0.5, 4.0), lo, hi)


@pytest.mark.parametrize("dtype,margin", [(np.float64, 1e-9), (np.float32, 1e-4)])
def test_containment_equals_convex_hull_of_the_vertices(oracle, dtype, margin):
    rng = np.random.default_rng(11)
    for trial in range(12):
        b = _frustum(rng)
        if trial % 2:                                        # clockwise listing must give the same solid
            b["xy_lo"], b["xy_hi"] = b["xy_lo"][::-1].copy(), b["xy_hi"][::-1].copy()
        lo64, hi64 = b["xy_lo"].astype(np.float64), b["xy_hi"].astype(np.float64)    # the float32 values, widened
        v = np.concatenate([np.c_[lo64, np.full(4, float(b["z_lo"]))], np.c_[hi64, np.full(4, float(b["z_hi"]))]])
        hull = ConvexHull(v)
        span = v.max(0) - v.min(0)
        pts = v.min(0) - 0.2 * span + rng.random((20000, 3)) * 1.4 * span
        # signed distance to the hull: max over facets of n.x + d (negative inside)
        dist = (pts @ hull.equations[:, :3].T + hull.equations[:, 3]).max(1)
        keep = np.abs(dist) > margin * (1 + np.abs(v).max())
        mat, _ = oracle.material_and_field(_geom([b]), pts, dtype=dtype)
        got = mat == 1
        assert 0.02 < got.mean() < 0.9
        assert np.array_equal(got[keep], dist[keep] < 0)
        assert keep.mean() > 0.99


def test_volume_matches_the_prismatoid_formula(oracle):
    # vertices move linearly in z, so the slice area is a quadratic in z and Simpson's rule is exact:
    # V = dz/6 (A_lo + 4 A_mid + A_hi), areas by the shoelace formula — also for a twisted (non-planar-sided) block
    rng = np.random.default_rng(12)

    def shoelace(q):
        x, y = q[:, 0], q[:, 1]
        return 0.5 * abs(np.dot(x, np.roll(y, -1)) - np.dot(y, np.roll(x, -1)))

    for trial in range(4):
        lo = _convex_quad(rng, (0.0, 0.0), (1.0, 1.5))
        hi = _convex_quad(rng, (0.3, -0.2), (1.4, 0.8)) if trial % 2 else lo * 0.5 + 0.25
        b = _block(-1.0, 2.0, lo, hi)
        lo64, hi64 = b["xy_lo"].astype(np.float64), b["xy_hi"].astype(np.float64)
        want = 3.0 / 6.0 * (shoelace(lo64) + 4 * shoelace(0.5 * (lo64 + hi64)) + shoelace(hi64))
        box_lo, box_hi = np.array([-2.5, -2.5, -1.0]), np.array([2.5, 2.5, 2.0])
        n = 400_000
        pts = box_lo + rng.random((n, 3)) * (box_hi - box_lo)
        mat, _ = oracle.material_and_field(_geom([b]), pts, dtype=np.float64)
        frac = (mat == 1).mean()
        box_v = np.prod(box_hi - box_lo)
        sigma = box_v * np.sqrt(frac * (1 - frac) / n)
        assert abs(frac * box_v - want) < 4 * sigma, (trial, frac * box_v, want, sigma)


def test_boxes_agree_with_the_region_lookup(oracle):
    regs = w.shield_regions(3)
    g_reg = Geometry(MODE_REGIONS, -1.0, 1.0, -1.0, 1.0, 0.0, 11.25, 1.0, 10, WORLD, regions=regs)
    g_pol = Geometry(MODE_POLY, -1.0, 1.0, -1.0, 1.0, 0.0, 11.25, 1.0, 10, WORLD, blocks=w.regions_as_blocks(regs))
    rng = np.random.default_rng(13)
    pts = np.array([-1.2, -1.2, -0.5]) + rng.random((100000, 3)) * np.array([2.4, 2.4, 12.5])
    for dtype in (np.float32, np.float64):
        m0, B0 = oracle.material_and_field(g_reg, pts, dtype=dtype)
        m1, B1 = oracle.material_and_field(g_pol, pts, dtype=dtype)
        assert np.array_equal(m0, m1) and np.array_equal(B0, B1)
    assert len(np.unique(m0)) == 3
    # z is half-open exactly as for regions; the lower z face belongs to the block, the upper one does not
    edge = np.array([[0.0, 0.0, 2.75], [0.0, 0.0, 0.0], [0.0, 0.0, 3.0], [0.0, 0.0, 3.5]], np.float32)
    m0, _ = oracle.material_and_field(g_reg, edge, dtype=np.float32)
    m1, _ = oracle.material_and_field(g_pol, edge, dtype=np.float32)
    assert np.array_equal(m0, m1)


def test_symmetries_first_block_wins_and_degenerate_slices(oracle):
    rng = np.random.default_rng(14)
    b = _frustum(rng)
    v_lo, v_hi = b["xy_lo"].copy(), b["xy_hi"].copy()
    pts = np.c_[rng.uniform(-4, 4, (50000, 2)), rng.uniform(float(b["z_lo"]) - 0.5, float(b["z_hi"]) + 0.5, 50000)]
    ref, _ = oracle.material_and_field(_geom([b]), pts, dtype=np.float32)
    # starting the vertex list elsewhere changes which edge is which, not the solid: same answer away from the boundary
    hull = ConvexHull(np.concatenate([np.c_[v_lo.astype(np.float64), np.full(4, float(b["z_lo"]))],
                                      np.c_[v_hi.astype(np.float64), np.full(4, float(b["z_hi"]))]]))
    off = np.abs((pts @ hull.equations[:, :3].T + hull.equations[:, 3]).max(1)) > 1e-4
    for k in (1, 2, 3):
        b2 = _block(b["z_lo"], b["z_hi"], np.roll(v_lo, k, 0), np.roll(v_hi, k, 0))
        m2, _ = oracle.material_and_field(_geom([b2]), pts, dtype=np.float32)
        assert np.array_equal(m2[off], ref[off])
    # overlapping blocks: the first in index order decides, field included
    big = _block(-10.0, 10.0, [(-5, -5), (5, -5), (5, 5), (-5, 5)], [(-5, -5), (5, -5), (5, 5), (-5, 5)], 2, (0.0, 1.0, 0.0))
    b["bx"] = 7.0
    m_ab, B_ab = oracle.material_and_field(_geom([b, big]), pts, dtype=np.float32)
    m_ba, B_ba = oracle.material_and_field(_geom([big, b]), pts, dtype=np.float32)
    assert np.array_equal(m_ab, np.where(ref == 1, 1, 2)) and np.all(m_ba == 2)
    assert np.array_equal(B_ab[:, 0], np.where(ref == 1, 7.0, 0.0).astype(np.float32)) and np.all(B_ba[:, 1] == 1.0)
    # pyramid: the lower face is a single point.  Its apex (a slice of zero area, every S_i = 0) contains nothing, and
    # so does a block whose slice has collapsed to a segment; a triangular prism (one repeated vertex) is a solid
    sq = [(-1, -1), (1, -1), (1, 1), (-1, 1)]
    pyr = _block(0.0, 1.0, [(0, 0)] * 4, sq)                  # apex at z = 0 (z_lo is inside the half-open range)
    q = np.array([[0.0, 0.0, 0.0], [0.3, 0.1, 0.0], [0.0, 0.0, 0.5], [0.49, -0.49, 0.5], [0.51, 0.0, 0.5]], np.float32)
    m, _ = oracle.material_and_field(_geom([pyr]), q, dtype=np.float32)
    assert m.tolist() == [WORLD, WORLD, 1, 1, WORLD]
    seg = _block(0.0, 1.0, [(-1, 0), (1, 0), (1, 0), (-1, 0)], [(-1, 0), (1, 0), (1, 0), (-1, 0)])
    m, _ = oracle.material_and_field(_geom([seg]), np.array([[0.0, 0.0, 0.5], [5.0, 0.0, 0.5]], np.float32), dtype=np.float32)
    assert np.all(m == WORLD)
    tri = _block(0.0, 1.0, [(0, 0), (2, 0), (0, 2), (0, 2)], [(0, 0), (2, 0), (0, 2), (0, 2)])
    tp = np.c_[rng.uniform(-0.5, 2.5, (20000, 2)), np.full(20000, 0.5)]
    m, _ = oracle.material_and_field(_geom([tri]), tp, dtype=np.float64)
    inside = (tp[:, 0] > 0) & (tp[:, 1] > 0) & (tp[:, 0] + tp[:, 1] < 2)
    assert np.array_equal(m == 1, inside)
    # NaN coordinates are outside
    m, _ = oracle.material_and_field(_geom([big]), np.array([[np.nan, 0, 0], [0, 0, np.nan]], np.float32), dtype=np.float32)
    assert np.all(m == WORLD)


def test_transport_through_box_blocks_equals_transport_through_regions(oracle):
    # whole-path pin: config 2's boxes written as polyhedra give the identical end state, bit for bit (the muons start
    # inside |x|,|y| < 0.5, away from every face, and a face hit exactly is a measure-zero event)
    wl = w.config2(n=3000, n_draws=20_000, n_cells=2)
    tabs = oracle.OracleTables(wl.hist)
    ref = oracle.transport(tabs, oracle.OracleGeometry(wl.geom), wl.muons.pos_q, wl.muons.mom, wl.seed, threads=4)
    g = wl.geom
    gp = Geometry(MODE_POLY, g.x_min, g.x_max, g.y_min, g.y_max, g.z_min, g.z_exit, g.p_min, g.max_steps,
                  g.world_material, blocks=w.regions_as_blocks(g.regions))
    got = oracle.transport(tabs, oracle.OracleGeometry(gp), wl.muons.pos_q, wl.muons.mom, wl.seed, threads=4)
    for k in ("flag", "steps", "pos", "mom"):
        assert np.array_equal(ref[k], got[k]), k
    assert len(np.unique(ref["flag"])) >= 2


def test_polyhedral_shield_workload_is_convex_and_bends_both_ways(oracle):
    blocks = w.shield_polyhedra(8)
    assert len(blocks) == 32
    for b in blocks:                                         # every face convex (cross products of one sign)
        for face in (b["xy_lo"].astype(np.float64), b["xy_hi"].astype(np.float64)):
            e = np.roll(face, -1, 0) - face
            cr = e[:, 0] * np.roll(e, -1, 0)[:, 1] - e[:, 1] * np.roll(e, -1, 0)[:, 0]
            assert np.all(cr > 0) or np.all(cr < 0)
    wl = w.config2p(n=2000, n_draws=20_000)
    # core and return yoke carry opposite fields; the gap between them is air
    m, B = oracle.material_and_field(wl.geom, np.array([[0.0, 0.0, 1.0], [0.5, 0.0, 1.0], [-0.5, 0.0, 1.0],
                                                         [0.335, 0.0, 1.0], [0.0, 0.0, 3.2], [0.0, 0.9, 1.0]], np.float32))
    assert m.tolist() == [1, 1, 1, 3, 2, 3]
    assert B[:, 1].tolist() == pytest.approx([1.7, -1.7, -1.7, 0.0, 0.0, 0.0])
    out = oracle.transport(oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom), wl.muons.pos_q, wl.muons.mom,
                           wl.seed, threads=4)
    assert set(np.unique(out["flag"])) >= {1, 3}
    assert out["steps"].max() <= 1700 and out["steps"].mean() > 200
