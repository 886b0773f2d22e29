"""Pins of the oracle's geometry and field lookups against
what the mathematics fixes: trilinear interpolation reproduces affine fields, returns the stored value at cell
centres and clamps at the faces; lookups agree with brute force, half-open on every boundary."""
import numpy as np

from paper_2512_10520_b200.workloads import Geometry, MODE_REGIONS, MODE_VOXEL, REGION_DTYPE, shield_regions


def _voxel(nx=7, ny=5, nz=9, cell=0.25, origin=(-1.0, 0.5, 2.0), field=None, material=None, world=3):
    rng = np.random.default_rng(1)
    field = rng.standard_normal((nz, ny, nx, 3)).astype(np.float32) if field is None else field
    material = rng.integers(0, 4, (nz, ny, nx)).astype(np.uint8) if material is None else material
    ox, oy, oz = origin
    return Geometry(MODE_VOXEL, -100.0, 100.0, -100.0, 100.0, -100.0, 100.0, 1.0, 10, world, nx=nx, ny=ny, nz=nz,
                    ox=ox, oy=oy, oz=oz, cell=cell, material=material, field=field)


def test_trilinear_reproduces_affine_fields(oracle):
    # B_c(r) = a_c + g_c . r sampled at cell centres; interior points (between the outermost centres) must
    # return the affine function itself: exactly in exact arithmetic, to rounding in double
    nx, ny, nz, cell, org = 7, 5, 9, 0.25, (-1.0, 0.5, 2.0)
    rng = np.random.default_rng(2)
    a, G = rng.standard_normal(3), rng.standard_normal((3, 3))
    zc, yc, xc = np.meshgrid(org[2] + (np.arange(nz) + 0.5) * cell, org[1] + (np.arange(ny) + 0.5) * cell,
                             org[0] + (np.arange(nx) + 0.5) * cell, indexing="ij")
    ctr = np.stack([xc, yc, zc], -1)
    fld = (a + ctr @ G.T)
    g = _voxel(nx, ny, nz, cell, org, field=fld.astype(np.float32))
    lo = np.array(org) + 0.5 * cell
    hi = np.array(org) + (np.array([nx, ny, nz]) - 0.5) * cell
    pts = lo + rng.random((5000, 3)) * (hi - lo)
    _, B = oracle.material_and_field(g, pts, dtype=np.float64)
    want = a + pts @ G.T
    assert np.abs(B - want).max() < 5e-6          # the stored field is float32; the interpolation adds ~1e-16
    # with a field exactly representable in float32 (small integers) the double-mode result is exact to 1e-12
    a2, G2 = np.array([1.0, -2.0, 3.0]), np.array([[4.0, 0, 0], [0, -8.0, 4.0], [8.0, 4.0, 0]])
    g2 = _voxel(nx, ny, nz, cell, org, field=(a2 + ctr @ G2.T).astype(np.float32))
    _, B2 = oracle.material_and_field(g2, pts, dtype=np.float64)
    assert np.abs(B2 - (a2 + pts @ G2.T)).max() < 1e-12


def test_trilinear_cell_centres_clamps_and_outside(oracle):
    g = _voxel()
    nx, ny, nz, cell = g.nx, g.ny, g.nz, g.cell
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    centres = np.stack([g.ox + (ix + 0.5) * cell, g.oy + (iy + 0.5) * cell, g.oz + (iz + 0.5) * cell], -1).reshape(-1, 3)
    mat, B = oracle.material_and_field(g, centres, dtype=np.float64)       # 0.25-m cells: centres are exact
    assert np.array_equal(B, g.field.reshape(-1, 3).astype(np.float64))
    assert np.array_equal(mat, g.material.reshape(-1))
    # within half a cell of a face the outer corner index is clamped: the field is constant along that axis
    p = np.array([[g.ox + 0.01, g.oy + 0.6, g.oz + 1.1], [g.ox + 0.12, g.oy + 0.6, g.oz + 1.1]])
    _, Bf = oracle.material_and_field(g, p, dtype=np.float64)
    assert np.allclose(Bf[0], Bf[1], rtol=0, atol=1e-15)
    # outside the grid (any axis, either side, and exactly on the upper face): world material, zero field
    out = np.array([[g.ox - 1e-3, g.oy + 0.1, g.oz + 0.1], [g.ox + nx * cell, g.oy + 0.1, g.oz + 0.1],
                    [g.ox + 0.1, g.oy - 1e-3, g.oz + 0.1], [g.ox + 0.1, g.oy + 0.1, g.oz + nz * cell + 5.0]])
    m, Bo = oracle.material_and_field(g, out, dtype=np.float32)
    assert np.all(m == g.world_material) and np.all(Bo == 0)
    # exactly on the lower faces: inside (half-open cells)
    m0, _ = oracle.material_and_field(g, np.array([[g.ox, g.oy, g.oz]]), dtype=np.float32)
    assert m0[0] == g.material[0, 0, 0]


def test_voxel_material_equals_numpy_floor(oracle):
    g = _voxel()
    rng = np.random.default_rng(3)
    pts = np.array([g.ox, g.oy, g.oz]) + rng.random((20000, 3)) * np.array([g.nx, g.ny, g.nz]) * g.cell
    pts = pts.astype(np.float32)
    inv = np.float32(1.0) / np.float32(g.cell)
    idx = np.floor((pts - np.array([g.ox, g.oy, g.oz], np.float32)) * inv).astype(int)
    ok = np.all((idx >= 0) & (idx < [g.nx, g.ny, g.nz]), axis=1)
    mat, _ = oracle.material_and_field(g, pts, dtype=np.float32)
    want = np.where(ok, g.material[np.clip(idx[:, 2], 0, g.nz - 1), np.clip(idx[:, 1], 0, g.ny - 1),
                                   np.clip(idx[:, 0], 0, g.nx - 1)], g.world_material)
    assert np.array_equal(mat, want)


def test_region_lookup_equals_brute_force(oracle):
    regs = shield_regions(8)
    g = Geometry(MODE_REGIONS, -1.0, 1.0, -1.0, 1.0, 0.0, 30.0, 1.0, 10, 3, regions=regs)
    rng = np.random.default_rng(4)
    pts = np.stack([rng.uniform(-1.1, 1.1, 40000), rng.uniform(-1.1, 1.1, 40000), rng.uniform(-0.5, 30.5, 40000)], 1)
    # points exactly on every boundary value of every region (z_lo, z_hi, x_lo, x_hi, y_lo, y_hi)
    edge = []
    for r in regs:
        for z in (r["z_lo"], r["z_hi"]):
            for x in (r["x_lo"], r["x_hi"], 0.0):
                for y in (r["y_lo"], r["y_hi"], 0.0):
                    edge.append((x, y, z))
    pts = np.concatenate([pts, np.array(edge)]).astype(np.float32)
    mat, B = oracle.material_and_field(g, pts, dtype=np.float32)
    want_m = np.full(len(pts), g.world_material, np.int32)
    want_B = np.zeros((len(pts), 3), np.float32)
    for r in regs:                                   # linear scan over all regions (z-disjoint: at most one hit)
        hit = ((pts[:, 2] >= r["z_lo"]) & (pts[:, 2] < r["z_hi"]) & (pts[:, 0] >= r["x_lo"]) & (pts[:, 0] < r["x_hi"])
               & (pts[:, 1] >= r["y_lo"]) & (pts[:, 1] < r["y_hi"]))
        want_m[hit] = r["material"]
        want_B[hit] = (r["bx"], r["by"], r["bz"])
    assert np.array_equal(mat, want_m) and np.array_equal(B, want_B)
    # no regions at all: world material everywhere
    g0 = Geometry(MODE_REGIONS, -1.0, 1.0, -1.0, 1.0, 0.0, 30.0, 1.0, 10, 2, regions=np.zeros(0, REGION_DTYPE))
    m0, B0 = oracle.material_and_field(g0, pts[:100], dtype=np.float32)
    assert np.all(m0 == 2) and np.all(B0 == 0)
