"""-m gpu: the convex-polyhedra geometry (§4.1, Eq. 2) of
the CUDA path against the oracle.  The library tests only the candidates its spatial hash lists for a point's cell, the
oracle scans every block: bit-exact agreement on dense random points — inside, outside, on faces and on hash-cell
boundaries — is what shows the pruning to be conservative, at every hash resolution."""
import numpy as np
import pytest

from gpu_util import compare, gpu_transport, ks_populations, oracle_transport

pytestmark = pytest.mark.gpu

WORLD = 3


def _lookup(mt, hist, geom, pts, hash_nxy=0, hash_nz=0):
    import torch
    b = mt.binding
    ctx = b.mt_create(0)
    try:
        b.mt_load_histograms(ctx, hist)
        b.mt_build_alias(ctx)
        b.mt_set_option(ctx, b.MT_OPT_HASH_NXY, hash_nxy)
        b.mt_set_option(ctx, b.MT_OPT_HASH_NZ, hash_nz)
        b.mt_set_geometry(ctx, geom)
        m, B = b.mt_debug_lookup(ctx, torch.from_numpy(np.ascontiguousarray(pts, np.float32)).cuda())
        torch.cuda.synchronize()
        return m.cpu().numpy(), B.cpu().numpy()
    finally:
        b.mt_destroy(ctx)


def _tiny_hist(n_materials=3):
    from paper_2512_10520_b200.workloads import Histograms
    M = n_materials
    one = np.ones((M, 2, 4), np.float32)
    ax = np.zeros((M, 2, 2), np.float32) + [-10.0, 0.5]
    return Histograms(M, 2, 4, 4, 1.0, 300.0, one, one.copy(), ax, ax.copy(), np.full(M + 1, 0.02, np.float32))


def _random_blocks(rng, n, world=2.0):
    from paper_2512_10520_b200.workloads import POLY_DTYPE
    out = np.zeros(n, POLY_DTYPE)
    for j in range(n):
        ang = np.sort(rng.uniform(0, 2 * np.pi, 4))
        while np.min(np.diff(np.concatenate([ang, [ang[0] + 2 * np.pi]]))) < 0.4:
            ang = np.sort(rng.uniform(0, 2 * np.pi, 4))
        c, r = rng.uniform(-world, world, 2), rng.uniform(0.1, 1.2, 2)
        lo = np.stack([c[0] + r[0] * np.cos(ang), c[1] + r[1] * np.sin(ang)], -1)
        hi = (lo - c) * rng.uniform(0.4, 1.6) + c + rng.uniform(-0.5, 0.5, 2)
        if j % 3 == 1:
            lo, hi = lo[::-1], hi[::-1]                       # clockwise
        if j % 7 == 3:
            hi[3] = hi[2]                                     # triangle on top
        if j % 11 == 5:
            hi[:] = hi.mean(0)                                # pyramid
        z0 = rng.uniform(0.0, 9.0)
        out[j]["z_lo"], out[j]["z_hi"] = z0, z0 + rng.uniform(0.05, 3.0)
        out[j]["xy_lo"], out[j]["xy_hi"] = lo, hi
        out[j]["material"] = 1 + j % 3
        out[j]["bx"], out[j]["by"], out[j]["bz"] = rng.standard_normal(3)
    return out


@pytest.mark.parametrize("hash_dims", [(0, 0), (1, 1), (3, 7), (64, 1024), (256, 50)])
def test_lookup_through_the_hash_equals_the_full_scan(mt, oracle, hash_dims):
    from paper_2512_10520_b200.workloads import Geometry, MODE_POLY
    rng = np.random.default_rng(21)
    blocks = _random_blocks(rng, 150)
    geom = Geometry(MODE_POLY, -2.0, 2.5, -2.0, 2.0, 0.0, 10.0, 1.0, 10, WORLD, blocks=blocks)
    n = 400_000
    pts = np.array([-2.6, -2.6, -0.5]) + rng.random((n, 3)) * np.array([5.7, 5.2, 11.5])      # also beyond the world box
    # points on block vertices, on the z faces, and on the hash grid's cell boundaries
    k = 0
    for b in blocks[:60]:
        for zf, face in ((b["z_lo"], b["xy_lo"]), (np.nextafter(b["z_hi"], np.float32(-1)), b["xy_hi"]), (b["z_hi"], b["xy_hi"])):
            for v in face:
                pts[k] = (v[0], v[1], zf); k += 1
    hx = max(hash_dims[0], 1) if hash_dims[0] else 16
    hz = max(hash_dims[1], 1) if hash_dims[1] else 256
    gx = (-2.0 + 4.5 * np.arange(hx + 1) / hx).astype(np.float32)
    gz = (10.0 * np.arange(hz + 1) / hz).astype(np.float32)
    m_edge = 20000
    pts[k:k + m_edge, 0] = rng.choice(gx, m_edge)
    pts[k + m_edge:k + 2 * m_edge, 2] = rng.choice(gz, m_edge)
    pts = pts.astype(np.float32)
    pts[-3:] = [[np.nan, 0, 1], [0, np.inf, 1], [0, 0, -np.inf]]
    m_ref, B_ref = oracle.material_and_field(geom, pts, dtype=np.float32)
    m_gpu, B_gpu = _lookup(mt, _tiny_hist(), geom, pts, *hash_dims)
    assert 0.05 < (m_ref != WORLD).mean() < 0.95
    assert np.array_equal(m_gpu, m_ref)
    assert np.array_equal(B_gpu.view(np.uint32), B_ref.view(np.uint32))


def test_debug_lookup_regions_and_voxel_modes(mt, oracle):
    # the same hook in the other two geometry modes (it is what the step loop calls)
    import torch
    from paper_2512_10520_b200 import workloads as w
    rng = np.random.default_rng(22)
    wl = w.config2(n=16, n_draws=2000, n_cells=3)
    pts = (np.array([-1.1, -1.1, -0.2]) + rng.random((100000, 3)) * np.array([2.2, 2.2, 11.6])).astype(np.float32)
    m_ref, B_ref = oracle.material_and_field(wl.geom, pts, dtype=np.float32)
    m_gpu, B_gpu = _lookup(mt, wl.hist, wl.geom, pts)
    assert np.array_equal(m_gpu, m_ref) and np.array_equal(B_gpu, B_ref)
    for field_mode in (0, 1):
        wl3 = w.config3(n=16, n_draws=2000, n_cells=1, half_width_cells=20, device="cuda", hist=wl.hist, field_mode=field_mode)
        g = wl3.geom
        lo = np.array([g.ox - 0.03, g.oy - 0.03, g.oz - 0.03])
        ext = np.array([g.nx, g.ny, g.nz]) * g.cell + 0.06
        pts = (lo + rng.random((200000, 3)) * ext).astype(np.float32)
        m_ref, B_ref = oracle.material_and_field(g, pts, dtype=np.float32)
        m_gpu, B_gpu = _lookup(mt, wl.hist, g, pts)
        assert np.array_equal(m_gpu, m_ref) and np.array_equal(B_gpu.view(np.uint32), B_ref.view(np.uint32))
        torch.cuda.empty_cache()


def _check(tag, g, ref, ks=False):
    c = compare(g, ref)
    print("%s: matched %.6f bit-exact %.6f max|dP|/P %.3g max|dr| %.3g" % (tag, c["matched"], c["bit_exact"], c["max_dp"], c["max_dr"]))
    assert c["matched"] >= 0.999 and c["bit_exact"] == 1.0
    if ks:
        assert all(p > 0.01 for p in ks_populations(g, ref).values())


def test_polyhedral_shield_transport_all_schedules(mt, oracle):
    from paper_2512_10520_b200 import workloads as w
    wl = w.config2p(n=100_000, n_draws=200_000)
    ref = oracle_transport(oracle, wl)
    assert set(np.unique(ref["flag"])) >= {1, 2, 3}
    for sched in (0, 1, 2, 3):
        g = gpu_transport(mt, wl, sched=sched)
        _check("config2p sched %d" % sched, g, ref, ks=(sched == 0))
        assert int(g["counters"][0]) == int(ref["steps"].sum())
    # ragged batch with an id offset, smaller blocks
    sel = np.arange(1000, 1000 + 33333)
    refs = oracle_transport(oracle, wl, sel=sel, id_base=5_000_000_000)
    _check("config2p ragged", gpu_transport(mt, wl, sel=sel, id_base=5_000_000_000, block=128), refs)


def test_polyhedral_shield_per_stage_field_and_joint_tables(mt, oracle):
    from paper_2512_10520_b200 import workloads as w
    wl = w.config2p(n=30_000, n_draws=100_000, field_mode=w.FIELD_PER_STAGE)
    ref = oracle_transport(oracle, wl)
    for sched in (2, 3):
        _check("config2p per-stage sched %d" % sched, gpu_transport(mt, wl, sched=sched), ref)
    frozen = oracle_transport(oracle, w.config2p(n=30_000, n_draws=100_000))
    assert not np.array_equal(frozen["pos"], ref["pos"])                 # the stage lookups cross block faces
    wj = w.config2p(n=30_000, n_draws=100_000, joint=True, table_shape=(20, 32, 16))
    _check("config2p joint", gpu_transport(mt, wj), oracle_transport(oracle, wj))


def test_box_blocks_reproduce_the_regions_geometry_on_the_gpu(mt, oracle):
    from paper_2512_10520_b200 import workloads as w
    from paper_2512_10520_b200.workloads import Geometry, MODE_POLY
    wl = w.config2(n=50_000, n_draws=100_000, n_cells=4)
    g_reg = gpu_transport(mt, wl)
    gm = wl.geom
    wl.geom = Geometry(MODE_POLY, gm.x_min, gm.x_max, gm.y_min, gm.y_max, gm.z_min, gm.z_exit, gm.p_min, gm.max_steps,
                       gm.world_material, blocks=w.regions_as_blocks(gm.regions))
    g_pol = gpu_transport(mt, wl)
    for k in ("flag", "steps", "pos", "mom"):
        assert np.array_equal(g_reg[k], g_pol[k]), k


def test_bad_blocks_are_refused(mt):
    from paper_2512_10520_b200.workloads import Geometry, MODE_POLY, POLY_DTYPE
    b = mt.binding
    sq = [(-1, -1), (1, -1), (1, 1), (-1, 1)]

    def blk(z_lo=0.0, z_hi=1.0, lo=sq, hi=sq, material=1):
        a = np.zeros(1, POLY_DTYPE)
        a[0]["z_lo"], a[0]["z_hi"], a[0]["xy_lo"], a[0]["xy_hi"], a[0]["material"] = z_lo, z_hi, lo, hi, material
        return a

    bad = [blk(z_lo=1.0, z_hi=1.0),                                       # empty z range
           blk(lo=[(-1, -1), (1, 1), (1, -1), (-1, 1)]),                  # self-intersecting (bow-tie) face
           blk(lo=[(-1, -1), (1, -1), (0.2, -0.5), (-1, 1)]),             # concave face
           blk(hi=sq[::-1]),                                              # faces in opposite orientations
           blk(material=9),
           blk(lo=[(np.nan, -1), (1, -1), (1, 1), (-1, 1)])]
    ctx = b.mt_create(0)
    try:
        b.mt_load_histograms(ctx, _tiny_hist())
        b.mt_build_alias(ctx)
        for blocks in bad:
            with pytest.raises(b.MtError) as e:
                b.mt_set_geometry(ctx, Geometry(MODE_POLY, -2.0, 2.0, -2.0, 2.0, 0.0, 2.0, 1.0, 10, WORLD, blocks=blocks))
            assert e.value.code == b.MT_ERR_INVALID_ARG
        with pytest.raises(b.MtError) as e:
            b.mt_set_geometry(ctx, Geometry(MODE_POLY, -2.0, 2.0, -2.0, 2.0, 0.0, 2.0, 1.0, 10, WORLD,
                                            blocks=np.repeat(blk(), 1025)))
        assert e.value.code == b.MT_ERR_UNSUPPORTED
        # an empty block list is a world of one material
        b.mt_set_geometry(ctx, Geometry(MODE_POLY, -2.0, 2.0, -2.0, 2.0, 0.0, 2.0, 1.0, 10, WORLD, blocks=np.zeros(0, POLY_DTYPE)))
    finally:
        b.mt_destroy(ctx)


def test_region_lookup_through_the_z_interval_table(mt, oracle):
    """The regions lookup (greatest j with z_lo[j] <= z, then the half-open box) goes through a z-cell
    table with two exact fix-up comparisons, or through the binary search when the intervals are too dense for the table;
    both against the oracle's search on points ON every z_lo / z_hi, one float either side, outside the world, NaN / inf."""
    from paper_2512_10520_b200.workloads import Geometry, MODE_REGIONS, REGION_DTYPE
    rng = np.random.default_rng(5)
    hist = _tiny_hist()

    def regions_from(z_edges, gap_every=3):
        regs = []
        for j, (a, b) in enumerate(zip(z_edges[:-1], z_edges[1:])):
            if gap_every and j % gap_every == 2:
                continue                                           # a hole: points there belong to the world
            regs.append((a, b, -0.5 + 0.1 * (j % 4), 0.6, -0.7, 0.4 + 0.05 * (j % 3), 1 + j % 2, 0.1 * j, -0.2, 0.01 * j))
        return np.array(regs, REGION_DTYPE)

    cases = {
        "uneven": np.sort(np.concatenate([[0.0, 30.0], rng.uniform(0.0, 30.0, 40)])).astype(np.float32),
        "two z_lo in one cell": np.array([0.0, 1.0, 2.0, 3.0, 4.0, 5.0, 5.004, 5.008, 10.0, 12.0, 14.0, 20.0, 20.011, 25.0,
                                          29.0, 30.0], np.float32),
        "dense (binary search)": np.linspace(2.0, 2.2, 1000).astype(np.float32),      # 0.2 mm intervals: no table possible
        "beyond the world box": np.array([-3.0, -1.0, 4.0, 31.0, 35.0, 36.0, 40.0], np.float32),
        "single": np.array([1.0, 2.0], np.float32),
        # the table is built from two regions on (the LEAN region kernels contain no search: MT_LEAN_ZTABLE)
        "two regions": np.array([1.0, 2.0, 7.5], np.float32),
        "three regions": np.array([0.0, 0.25, 29.0, 30.0], np.float32),
    }
    for name, z_edges in cases.items():
        z_edges = np.unique(z_edges)
        regs = regions_from(z_edges, gap_every=0 if name in ("single", "dense (binary search)", "two z_lo in one cell", "two regions", "three regions") else 3)
        geom = Geometry(MODE_REGIONS, -1.0, 1.0, -1.0, 1.0, 0.0, 30.0, 1.0, 100, 2, regions=regs)
        zs = np.concatenate([regs["z_lo"], regs["z_hi"]])
        special = np.concatenate([zs, np.nextafter(zs, np.float32(-np.inf)), np.nextafter(zs, np.float32(np.inf)),
                                  np.float32([-1e30, -5.0, 0.0, 30.0, 45.0, 1e30, np.nan, np.inf, -np.inf])])
        n = 60000
        pts = np.empty((n, 3), np.float32)
        pts[:, 0] = rng.uniform(-0.8, 0.8, n)
        pts[:, 1] = rng.uniform(-0.9, 0.7, n)
        pts[:, 2] = np.where(rng.random(n) < 0.5, rng.choice(special, n), rng.uniform(-4.0, 42.0, n).astype(np.float32))
        pts[::7, 0] = rng.choice(np.float32([-0.5, -0.4, 0.6]), len(pts[::7]))     # on x faces
        m_ref, B_ref = oracle.material_and_field(geom, pts, dtype=np.float32)
        m_gpu, B_gpu = _lookup(mt, hist, geom, pts)
        assert (m_ref != 2).mean() > 0.02, name
        assert np.array_equal(m_gpu, m_ref), name
        assert np.array_equal(B_gpu.view(np.uint32), B_ref.view(np.uint32)), name
