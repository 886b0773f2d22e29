"""-m gpu: the LEAN kernel variant — the wavefront voxel kernel with the operations dropped that the host
has proven to be identities for the loaded tables and geometry — against the oracle and against the general kernels,
bit for bit, including the floats next to a face of the world box that map outside the grid and therefore leave the
proven interval."""
import numpy as np
import pytest

from gpu_util import compare, gpu_transport, oracle_transport, unpack

pytestmark = pytest.mark.gpu


def _run(mt, wl, no_lean, pos_q=None, mom=None):
    import torch
    b = mt.binding
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        h.set_option(b.MT_OPT_NO_LEAN, no_lean)
        pos_q = wl.muons.pos_q if pos_q is None else pos_q
        mom = wl.muons.mom if mom is None else mom
        out = h.transport(torch.from_numpy(np.ascontiguousarray(pos_q)).cuda(), torch.from_numpy(np.ascontiguousarray(mom)).cuda(), wl.seed)
        torch.cuda.synchronize()
        info = {k: b.mt_get_info(h.ctx, v) for k, v in (("facts", b.MT_INFO_LEAN_FACTS), ("lean", b.MT_INFO_LAST_LEAN),
                                                       ("sched", b.MT_INFO_LAST_SCHEDULE))}
        return unpack(out["pos_flag"].cpu().numpy(), out["mom_steps"].cpu().numpy()), info
    finally:
        h.close()


def test_lean_variant_runs_and_matches_oracle_and_general_kernel(mt, oracle):
    from paper_2512_10520_b200 import workloads as w
    wl = w.config3(n=60_000, n_draws=200_000, n_cells=2, half_width_cells=40, device="cuda")
    lean, info = _run(mt, wl, 0)
    assert info == {"facts": 3, "lean": 1, "sched": 3}
    gen, info2 = _run(mt, wl, 1)
    assert info2["lean"] == 0
    for k in ("flag", "steps", "pos", "mom"):
        assert np.array_equal(lean[k], gen[k]), k
    ref = oracle_transport(oracle, wl)
    c = compare(lean, ref)
    assert c["bit_exact"] == 1.0 and c["matched"] >= 0.999
    assert set(np.unique(ref["flag"])) >= {2, 3}


def test_lean_variant_on_the_faces_of_the_world_box_and_odd_momenta(mt, oracle):
    # 0.4 - 2^-25 is inside the world box (x < 0.4) but (x + 0.4) * 100 rounds to 80 = nx: outside the grid, world
    # material, no field — the lean kernel must hand such lanes to the general code.  Same for y and z, the lower faces,
    # and momenta outside the fast path's range.
    from paper_2512_10520_b200 import workloads as w
    wl = w.config3(n=4096, n_draws=50_000, n_cells=1, half_width_cells=40, device="cuda")
    g = wl.geom
    f32 = np.float32
    below = lambda v: np.nextafter(f32(v), f32(-np.inf))
    above = lambda v: np.nextafter(f32(v), f32(np.inf))
    pos_q, mom = wl.muons.pos_q.copy(), wl.muons.mom.copy()
    specials = [(below(g.x_max), 0.0, 0.5), (0.0, below(g.y_max), 0.5), (g.x_min, g.y_min, 0.0), (above(g.x_min), 0.1, 1.0),
                (0.1, 0.1, below(g.z_exit)), (below(below(g.x_max)), below(below(g.y_max)), 2.0), (g.x_max, 0.0, 1.0),
                (0.0, 0.0, g.z_exit), (np.nan, 0.0, 1.0), (0.0, np.nan, 1.0), (0.0, 0.0, np.nan), (0.0, 0.0, -1e-30)]
    for k, (x, y, z) in enumerate(specials):
        pos_q[k, :3] = (x, y, z)
        mom[k, :3] = (0.0, 0.0, 20.0)
    n0 = len(specials)
    mom[n0 + 0, :3] = (0.0, 0.0, 0.0)
    mom[n0 + 1, :3] = (np.nan, 1.0, 1.0)
    mom[n0 + 2, :3] = (1e30, 1e30, 1e30)
    mom[n0 + 3, :3] = (0.0, 0.0, 1e-30)
    mom[n0 + 4, :3] = (np.inf, 0.0, 1.0)
    # sideways and backwards movers that leave through every face
    mom[n0 + 5, :3] = (30.0, 0.0, 0.1)
    mom[n0 + 6, :3] = (-30.0, 0.0, 0.1)
    mom[n0 + 7, :3] = (0.0, 30.0, 0.1)
    mom[n0 + 8, :3] = (0.0, -30.0, 0.1)
    mom[n0 + 9, :3] = (0.0, 0.1, -30.0)
    wl.muons.pos_q, wl.muons.mom = pos_q, mom
    lean, info = _run(mt, wl, 0)
    assert info["lean"] == 1
    gen, _ = _run(mt, wl, 1)
    ref = oracle_transport(oracle, wl)
    for k in ("flag", "steps"):
        assert np.array_equal(lean[k], ref[k]) and np.array_equal(gen[k], ref[k]), k
    for k in ("pos", "mom"):                       # bit for bit, except that a NaN may carry another payload
        for got in (lean[k], gen[k]):
            nan = np.isnan(ref[k])
            assert np.array_equal(np.isnan(got), nan), k
            assert np.array_equal(got.view(np.uint32)[~nan], ref[k].view(np.uint32)[~nan]), k
    # the face floats did take a step (they are inside the world box) in the world material
    assert ref["steps"][0] > 0 and ref["steps"][1] > 0 and ref["flag"][6] == 3 and ref["steps"][6] == 0


def test_lean_facts_are_refused_when_an_axis_reaches_a_clamp(mt, oracle):
    # a Dp/p axis that reaches above log2(0.999): the cap on f is live, the lean variant must not be taken
    from paper_2512_10520_b200 import workloads as w
    wl = w.config3(n=20_000, n_draws=50_000, n_cells=1, half_width_cells=20, device="cuda")
    wl.hist.axis_dp = wl.hist.axis_dp.copy()
    wl.hist.axis_dp[0, :, 0] = -6.0          # iron: f from 2^-6 up to 2^(-6 + 256 * d)
    wl.hist.axis_dp[0, :, 1] = 0.03          # -6 + 7.68 = 1.68 > 0: f is capped at 0.999 for the top cells
    got, info = _run(mt, wl, 0)
    assert info["facts"] == 2 and info["lean"] == 0
    ref = oracle_transport(oracle, wl)
    c = compare(got, ref)
    assert c["bit_exact"] == 1.0


@pytest.mark.parametrize("joint,field_mode", [(False, 1), (False, 2), (False, 3), (True, 0), (True, 2)])
def test_lean_variants_of_the_other_voxel_modes(mt, oracle, joint, field_mode):
    # nearest-neighbour / per-stage field and the joint 2D tables have lean kernels too (the stage lookups keep their
    # inside test: a stage position may lie outside the grid)
    from paper_2512_10520_b200 import workloads as w
    shape = (20, 32, 16) if joint else (100, 256, 128)
    wl = w.config3(n=20_000, n_draws=100_000, n_cells=1, half_width_cells=30, device="cuda", joint=joint,
                   table_shape=shape, field_mode=field_mode)
    lean, info = _run(mt, wl, 0)
    assert info["facts"] == 3 and info["lean"] == 1
    gen, info2 = _run(mt, wl, 1)
    assert info2["lean"] == 0
    ref = oracle_transport(oracle, wl)
    for got in (lean, gen):
        c = compare(got, ref)
        assert c["bit_exact"] == 1.0 and c["matched"] >= 0.999


@pytest.mark.parametrize("which,sched", [("config1", 0), ("config2", 0), ("config2", 3), ("config2p", 0), ("config2p", 2),
                                         ("config2_joint", 0), ("config2p_per_stage", 0), ("config2_few_regions", 2),
                                         ("config2_few_regions", 3)])
def test_lean_variants_of_regions_and_polyhedra(mt, oracle, which, sched):
    # regions and polyhedra take the lean kernels on the table facts alone (clamps, caps, theta < pi/4): REFILL and
    # WAVEFRONT, tables from L2 or (config 1: 38 KB) staged in shared memory
    import torch
    from paper_2512_10520_b200 import workloads as w
    b = mt.binding
    wl = {"config1": lambda: w.config1(n=20_000, n_draws=100_000),
          "config2": lambda: w.config2(n=40_000, n_draws=100_000, n_cells=4),
          # one cell of the shield: a handful of regions, for which the z-interval table is built too (the LEAN region
          # kernels contain no binary search: MT_LEAN_ZTABLE)
          "config2_few_regions": lambda: w.config2(n=20_000, n_draws=100_000, n_cells=1),
          "config2p": lambda: w.config2p(n=40_000, n_draws=100_000, n_cells=4),
          "config2_joint": lambda: w.config2(n=20_000, n_draws=100_000, n_cells=2, joint=True, table_shape=(20, 32, 16)),
          "config2p_per_stage": lambda: w.config2p(n=20_000, n_draws=100_000, n_cells=2, field_mode=w.FIELD_PER_STAGE)}[which]()
    ref = oracle_transport(oracle, wl)
    for no_lean in (0, 1):
        h = b.MuonTransport(0).setup(wl.hist, wl.geom)
        try:
            h.set_option(b.MT_OPT_NO_LEAN, no_lean).set_option(b.MT_OPT_SCHEDULE, sched)
            out = h.transport(torch.from_numpy(wl.muons.pos_q).cuda(), torch.from_numpy(wl.muons.mom).cuda(), wl.seed)
            torch.cuda.synchronize()
            assert b.mt_get_info(h.ctx, b.MT_INFO_LEAN_FACTS) & 1
            assert b.mt_get_info(h.ctx, b.MT_INFO_LAST_LEAN) == 1 - no_lean
            got = unpack(out["pos_flag"].cpu().numpy(), out["mom_steps"].cpu().numpy())
        finally:
            h.close()
        c = compare(got, ref)
        assert c["bit_exact"] == 1.0 and c["matched"] >= 0.999


def test_lean_region_kernels_are_refused_when_no_z_interval_table_exists(mt, oracle):
    # 1000 slabs of 0.2 mm: more than two z_lo per table cell at any table size, so the lookup has to search — which only the
    # general kernels contain (MT_LEAN_ZTABLE is part of the facts a LEAN region kernel needs)
    import copy
    import torch
    from paper_2512_10520_b200 import workloads as w
    b = mt.binding
    wl = w.config1(n=8192, n_draws=100_000)
    edges = np.linspace(2.0, 2.2, 1001).astype(np.float32)
    regs = np.array([(a, c, -1.0, 1.0, -1.0, 1.0, 1, 0.0, 1.7 * (1 - 2 * (j & 1)), 0.0)
                     for j, (a, c) in enumerate(zip(edges[:-1], edges[1:])) if c > a], w.REGION_DTYPE)
    geom = copy.copy(wl.geom)
    geom.regions = regs
    wl = copy.copy(wl)
    wl.geom = geom
    ref = oracle_transport(oracle, wl)
    for sched in (2, 3):
        h = b.MuonTransport(0).setup(wl.hist, wl.geom)
        try:
            h.set_option(b.MT_OPT_SCHEDULE, sched)
            out = h.transport(torch.from_numpy(wl.muons.pos_q).cuda(), torch.from_numpy(wl.muons.mom).cuda(), wl.seed)
            torch.cuda.synchronize()
            assert b.mt_get_info(h.ctx, b.MT_INFO_LEAN_FACTS) & 1            # the table axes would allow it
            assert b.mt_get_info(h.ctx, b.MT_INFO_LAST_LEAN) == 0
            got = unpack(out["pos_flag"].cpu().numpy(), out["mom_steps"].cpu().numpy())
        finally:
            h.close()
        c = compare(got, ref)
        assert c["bit_exact"] == 1.0 and c["matched"] >= 0.999
