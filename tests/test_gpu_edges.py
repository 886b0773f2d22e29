"""-m gpu: launch independence (P-12), edge cases, exit records, the host-buffer call and error behaviour."""
import numpy as np
import pytest

from gpu_util import compare, gpu_transport, oracle_transport, unpack

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def wl1(workloads):
    return workloads.config1(n=20_000, n_draws=100_000)


@pytest.fixture(scope="module")
def ref1(oracle, wl1):
    return oracle_transport(oracle, wl1)


def _same(a, b):
    return all(np.array_equal(a[k].view(np.uint32) if a[k].dtype == np.float32 else a[k],
                              b[k].view(np.uint32) if b[k].dtype == np.float32 else b[k]) for k in ("pos", "mom", "flag", "steps"))


def test_results_do_not_depend_on_launch_shape(mt, wl1, ref1):
    base = gpu_transport(mt, wl1, sched=1, block=256)
    assert compare(base, ref1)["bit_exact"] == 1.0
    for kw in (dict(sched=1, block=32), dict(sched=2, block=64, min_idle=1), dict(sched=2, block=256, min_idle=16),
               dict(sched=2, block=128, min_idle=32), dict(sched=3, block=96, slab=10), dict(sched=3, slab=1000),
               dict(sched=2, placement=2), dict(sched=2, placement=1),
               # concurrent lanes (contiguous id ranges on the library's own streams): ragged last lane, more lanes than fit
               dict(sched=3, lanes=2), dict(sched=3, lanes=7, slab=30), dict(sched=2, lanes=3), dict(sched=1, lanes=16),
               # WAVEFRONT pass modes: persistent CTAs / one item per warp, with either lane-priority scheme and odd blocks
               dict(sched=3, lanes=1, pass_mode=2), dict(sched=3, lanes=3, pass_mode=2, block=96, lane_prio=1),
               dict(sched=3, lanes=4, pass_mode=1, lane_prio=2), dict(sched=3, lanes=5, pass_mode=2, block=32, slab=17),
               # the live list re-sorted only after every k-th pass
               dict(sched=3, slab=20, sort_every=2), dict(sched=3, slab=7, sort_every=5, lanes=2), dict(sched=3, slab=20, sort_every=64)):
        assert _same(gpu_transport(mt, wl1, **kw), base), kw


def test_batch_split_and_permutation(mt, oracle, wl1, ref1):
    n = len(wl1.muons.pos_q)
    # split into ragged batches with id_base: identical to the single call
    cuts = [0, 1, 34, 5000, 5000, 12345, n]
    parts = [gpu_transport(mt, wl1, sel=slice(a, b), id_base=a) for a, b in zip(cuts[:-1], cuts[1:]) if b > a]
    for k in ("pos", "mom", "flag", "steps"):
        assert np.array_equal(np.concatenate([p[k] for p in parts]), ref1[k])
    # ids offset: muon j of the call gets id id_base + j
    g = gpu_transport(mt, wl1, id_base=2 ** 33 + 7)
    r = oracle_transport(oracle, wl1, id_base=2 ** 33 + 7)
    assert compare(g, r)["bit_exact"] == 1.0
    assert not np.array_equal(g["mom"], ref1["mom"])


def test_ragged_and_tiny_sizes(mt, oracle, wl1):
    for n in (1, 31, 32, 33, 257):
        g = gpu_transport(mt, wl1, sel=slice(0, n), sched=2)
        r = oracle_transport(oracle, wl1, sel=slice(0, n))
        assert compare(g, r)["bit_exact"] == 1.0
    # n = 0 is a no-op
    import torch
    b = mt.binding
    h = b.MuonTransport(0).setup(wl1.hist, wl1.geom)
    try:
        out = h.transport(torch.zeros((0, 4), device="cuda"), torch.zeros((0, 4), device="cuda"), 1)
        assert out["pos_flag"].shape == (0, 4)
    finally:
        h.close()


def test_degenerate_muons(mt, oracle, workloads):
    """Already below the cut, already past the exit plane, outside the world, NaN momentum, pointing at -z,
    zero step budget; and vacuum-only flight is a straight line (P-5)."""
    import copy
    wl = workloads.config1(n=8, n_draws=50_000)
    wl = copy.deepcopy(wl)
    pq, mo = wl.muons.pos_q, wl.muons.mom
    pq[:] = 0.0
    pq[:, 3] = 1.0
    mo[:] = 0.0
    mo[:, 2] = 20.0
    mo[0, 2] = 0.5                      # below p_min -> STOPPED at step 0
    pq[1, 2] = 6.0                      # on the exit plane -> EXITED at step 0
    pq[2, 0] = 1.0                      # x == x_max -> ESCAPED
    pq[3, 2] = -0.001                   # z < z_min -> ESCAPED
    mo[4, 2] = np.nan                   # NaN -> STOPPED
    mo[5] = (0.0, 0.0, -20.0, 0.0)      # heading -z from z = 0: leaves through z_min
    pq[5, 2] = 0.05
    mo[6] = (19.0, 0.0, 3.0, 0.0)       # steep: lateral escape
    g = gpu_transport(mt, wl, sched=2)
    r = oracle_transport(oracle, wl)
    assert np.array_equal(g["flag"], r["flag"]) and np.array_equal(g["steps"], r["steps"])
    assert list(g["flag"][:5]) == [1, 2, 3, 3, 1] and list(g["steps"][:5]) == [0, 0, 0, 0, 0]
    ok = ~np.isnan(r["mom"]).any(axis=1)
    assert np.array_equal(g["pos"][ok], r["pos"][ok]) and np.array_equal(g["mom"][ok], r["mom"][ok])
    # max_steps = 0 -> everything still alive is MAXSTEPS at step 0
    wl.geom.max_steps = 0
    g = gpu_transport(mt, wl, sched=1)
    assert list(g["flag"][5:8]) == [4, 4, 4] and np.all(g["steps"] == 0)
    # vacuum world, no regions: straight line, momentum untouched, no random numbers drawn
    wl2 = workloads.config0(n=64, n_draws=50_000)
    wl2.geom.regions = wl2.geom.regions[:0]
    wl2.muons.mom[:, 0] = np.linspace(-5, 5, 64)
    g = gpu_transport(mt, wl2, sched=2)
    r = oracle_transport(oracle, wl2)
    assert compare(g, r)["bit_exact"] == 1.0
    assert np.array_equal(g["mom"], wl2.muons.mom[:, :3])
    d = wl2.muons.mom[:, :3].astype(np.float64)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    h = float(wl2.hist.step_m[0])
    assert np.abs(g["pos"] - g["steps"][:, None] * h * d).max() < 2e-5


def test_exit_records_and_counters(mt, wl1, ref1):
    n = len(ref1["flag"])
    n_exit = int((ref1["flag"] == 2).sum())
    g = gpu_transport(mt, wl1, sched=2, exit_capacity=n)
    assert g["exit_count"] == n_exit
    rec = g["exit_rec"][:n_exit]
    idx = rec[:, 3].copy().view(np.uint32)
    assert len(np.unique(idx)) == n_exit and np.array_equal(np.sort(idx), np.nonzero(ref1["flag"] == 2)[0])
    assert np.array_equal(rec[:, :3], ref1["pos"][idx]) and np.array_equal(rec[:, 4:7], ref1["mom"][idx])
    assert np.array_equal(rec[:, 7].copy().view(np.int32), ref1["steps"][idx])
    # lanes: the records carry the index within the CALL, not within the lane
    for sched in (2, 3):
        g = gpu_transport(mt, wl1, sched=sched, exit_capacity=n, lanes=5)
        assert g["exit_count"] == n_exit
        rec = g["exit_rec"][:n_exit]
        idx = rec[:, 3].copy().view(np.uint32)
        assert np.array_equal(np.sort(idx), np.nonzero(ref1["flag"] == 2)[0])
        assert np.array_equal(rec[:, :3], ref1["pos"][idx]) and np.array_equal(rec[:, 4:7], ref1["mom"][idx])
    # capacity smaller than the number of hits: the count still reports all, only `capacity` records are written
    g = gpu_transport(mt, wl1, sched=3, exit_capacity=100)
    assert g["exit_count"] == n_exit
    idx = g["exit_rec"][:, 3].copy().view(np.uint32)
    assert np.all(ref1["flag"][idx] == 2)
    assert g["counters"][0] == ref1["steps"].sum()
    assert np.array_equal(g["counters"][1:5], np.bincount(ref1["flag"], minlength=5)[1:5])


@pytest.mark.parametrize("sched", [1, 2, 3])
def test_exit_records_projected_onto_the_plane(mt, oracle, wl1, ref1, sched):
    # with MT_EXIT_PROJECT the compact list holds the oracle's projection of every EXITED muon, bit for
    # bit; the dense outputs stay the state at the break
    import copy
    wl = copy.copy(wl1)
    wl.geom = copy.copy(wl1.geom)
    wl.geom.exit_mode = 1
    n = len(ref1["flag"])
    hit = np.nonzero(ref1["flag"] == 2)[0]
    g = gpu_transport(mt, wl, sched=sched, exit_capacity=n)
    assert g["exit_count"] == len(hit)
    for k in ("pos", "mom", "flag", "steps"):
        assert np.array_equal(g[k], ref1[k]), k
    rec = g["exit_rec"][:len(hit)]
    idx = rec[:, 3].copy().view(np.uint32)
    assert np.array_equal(np.sort(idx), hit)
    want = oracle.exit_project(ref1["pos"][idx], ref1["mom"][idx], wl.geom.z_exit, dtype=np.float32)
    assert np.array_equal(rec[:, :3].view(np.uint32), want.view(np.uint32))
    assert np.all(rec[:, 2] == np.float32(wl.geom.z_exit)) and np.any(ref1["pos"][idx][:, 2] > wl.geom.z_exit)
    assert np.array_equal(rec[:, 4:7], ref1["mom"][idx])
    # the projection moved the points by up to a step's worth of transverse travel
    moved = np.abs(rec[:, :2] - ref1["pos"][idx][:, :2]).max()
    assert 1e-5 < moved < 0.02


def test_host_buffer_call(mt, wl1, ref1):
    import torch
    b = mt.binding
    h = b.MuonTransport(0).setup(wl1.hist, wl1.geom)
    try:
        out = h.transport_host(wl1.muons.pos_q, wl1.muons.mom, wl1.seed, exit_capacity=64)
        g = unpack(out["pos_flag"], out["mom_steps"])
        assert compare(g, ref1)["bit_exact"] == 1.0
        assert out["counters"][0] == ref1["steps"].sum() and out["exit_count"][0] == (ref1["flag"] == 2).sum()
        # lanes copy their own ranges in and out
        h.set_option(b.MT_OPT_LANES, 3)
        out = h.transport_host(wl1.muons.pos_q, wl1.muons.mom, wl1.seed, exit_capacity=64)
        assert compare(unpack(out["pos_flag"], out["mom_steps"]), ref1)["bit_exact"] == 1.0
        assert out["counters"][0] == ref1["steps"].sum() and out["exit_count"][0] == (ref1["flag"] == 2).sum()
        assert b.mt_get_info(h.ctx, b.MT_INFO_LAST_LANES) == 3
        # pinned torch tensors work too
        pq = torch.from_numpy(wl1.muons.pos_q).pin_memory()
        mo = torch.from_numpy(wl1.muons.mom).pin_memory()
        o = dict(pos_flag=torch.empty((len(pq), 4)).pin_memory(), mom_steps=torch.empty((len(pq), 4)).pin_memory())
        h.transport_host(pq, mo, wl1.seed, out=o)
        assert compare(unpack(o["pos_flag"].numpy(), o["mom_steps"].numpy()), ref1)["bit_exact"] == 1.0
    finally:
        h.close()


def test_error_behaviour(mt, workloads):
    import copy
    b = mt.binding
    wl = workloads.config0(n=8, n_draws=20_000)
    ctx = b.mt_create(0)
    try:
        with pytest.raises(b.MtError) as e:
            b.mt_build_alias(ctx)
        assert e.value.code == b.MT_ERR_STATE
        b.mt_load_histograms(ctx, wl.hist)
        with pytest.raises(b.MtError) as e:
            b.mt_set_geometry(ctx, wl.geom)
        assert e.value.code == b.MT_ERR_STATE
        bad = copy.deepcopy(wl.hist)
        bad.counts_th[0, 7, :] = 0.0
        b.mt_load_histograms(ctx, bad)
        with pytest.raises(b.MtError) as e:
            b.mt_build_alias(ctx)
        assert e.value.code == b.MT_ERR_EMPTY_HIST and "bin 7" in str(e.value)
        b.mt_load_histograms(ctx, wl.hist)
        b.mt_build_alias(ctx)
        g = copy.deepcopy(wl.geom)
        g.regions = np.concatenate([g.regions, g.regions])        # overlapping in z
        with pytest.raises(b.MtError) as e:
            b.mt_set_geometry(ctx, g)
        assert e.value.code == b.MT_ERR_INVALID_ARG
        with pytest.raises(b.MtError) as e:
            b.mt_set_option(ctx, b.MT_OPT_BLOCK_THREADS, 100)
        assert e.value.code == b.MT_ERR_INVALID_ARG
    finally:
        b.mt_destroy(ctx)
    with pytest.raises(b.MtError):
        b.mt_create(9999)


def test_reloading_histograms_invalidates_tables_and_geometry(mt, oracle, workloads):
    """load -> build -> set_geometry -> load(new shape) must not transport against the old tables / blob."""
    import torch
    b = mt.binding
    wl = workloads.config1(n=512, n_draws=30_000)
    other = workloads.make_histograms(0, ["iron", "concrete"], [2.0, 2.0], 20, 1.0, 300.0, 32, 16, 20_000)
    dq, dm = torch.from_numpy(wl.muons.pos_q).cuda(), torch.from_numpy(wl.muons.mom).cuda()
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        h.transport(dq, dm, wl.seed)
        b.mt_load_histograms(h.ctx, other)                       # new shape: 2 materials, 20 bins, 32 + 16 cells
        for call in (lambda: h.transport(dq, dm, wl.seed),
                     lambda: h.transport_host(wl.muons.pos_q, wl.muons.mom, wl.seed),
                     lambda: b.mt_debug_lookup(h.ctx, torch.zeros((4, 3), device="cuda"))):
            with pytest.raises(b.MtError) as e:
                call()
            assert e.value.code == b.MT_ERR_STATE
        b.mt_build_alias(h.ctx)
        with pytest.raises(b.MtError) as e:                      # tables rebuilt, geometry still missing
            h.transport(dq, dm, wl.seed)
        assert e.value.code == b.MT_ERR_STATE
        b.mt_set_geometry(h.ctx, wl.geom)
        wl2 = workloads.Workload("reloaded", other, wl.geom, wl.muons, seed=wl.seed)
        out = h.transport(dq, dm, wl.seed)
        torch.cuda.synchronize()
        g = unpack(out["pos_flag"].cpu().numpy(), out["mom_steps"].cpu().numpy())
        assert compare(g, oracle_transport(oracle, wl2))["bit_exact"] == 1.0
        # mt_build_alias again with a geometry in place keeps it (and the results)
        b.mt_build_alias(h.ctx, b.MT_PLACE_L2)
        out = h.transport(dq, dm, wl.seed)
        torch.cuda.synchronize()
        assert compare(unpack(out["pos_flag"].cpu().numpy(), out["mom_steps"].cpu().numpy()), g)["bit_exact"] == 1.0
    finally:
        h.close()


def test_failed_voxel_geometry_leaves_no_geometry(mt, workloads):
    """mt_set_geometry(VOXEL) overwrites the library's grid before it can validate the material ids; on
    failure the context must not keep transporting with the old parameters over the new data."""
    import copy
    import torch
    b = mt.binding
    wl = workloads.config3(n=256, n_draws=20_000, n_cells=1, half_width_cells=16, device="cuda")
    dq, dm = torch.from_numpy(wl.muons.pos_q).cuda(), torch.from_numpy(wl.muons.mom).cuda()
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        h.transport(dq, dm, wl.seed)
        bad = copy.copy(wl.geom)
        bad.material = wl.geom.material.clone()
        bad.material[3, 3, 3] = 9                                # > n_materials = 3
        with pytest.raises(b.MtError) as e:
            b.mt_set_geometry(h.ctx, bad)
        assert e.value.code == b.MT_ERR_INVALID_ARG
        with pytest.raises(b.MtError) as e:
            h.transport(dq, dm, wl.seed)
        assert e.value.code == b.MT_ERR_STATE
        # an argument error caught before the grid is touched keeps a geometry that is set
        b.mt_set_geometry(h.ctx, wl.geom)
        bad2 = copy.copy(wl.geom)
        bad2.cell = -1.0
        with pytest.raises(b.MtError):
            b.mt_set_geometry(h.ctx, bad2)
        h.transport(dq, dm, wl.seed)
        torch.cuda.synchronize()
    finally:
        h.close()


def test_exit_count_without_a_list(mt, wl1, ref1):
    """include/muon_transport.h: exit_count may be given alone; it counts every EXITED muon."""
    import torch
    b = mt.binding
    h = b.MuonTransport(0).setup(wl1.hist, wl1.geom)
    try:
        dq, dm = torch.from_numpy(wl1.muons.pos_q).cuda(), torch.from_numpy(wl1.muons.mom).cuda()
        for sched in (1, 2, 3):
            h.set_option(b.MT_OPT_SCHEDULE, sched)
            side = torch.cuda.Stream()                           # zero-fills and kernels on a non-current stream
            out = h.transport(dq, dm, wl1.seed, count_exits=True, stream=side)
            side.synchronize()
            assert "exit_rec" not in out and int(out["exit_count"].item()) == int((ref1["flag"] == 2).sum())
            assert int(out["counters"][0].item()) == int(ref1["steps"].sum())
    finally:
        h.close()
