"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances are north_star's: sampled indices bit-exact; per muon |dP|/P <= 1e-5, |dr| <= 1e-5 m, same flag and
step count on >= 99.9 % of muons; KS p > 0.01 on final p, theta, x, y.  Because both sides evaluate the same
float32 contract the tests also report — and require — the bit-exact fraction.
"""
import functools

import numpy as np
import pytest

from gpu_util import compare, gpu_transport, ks_populations, need_device_memory, oracle_transport

pytestmark = pytest.mark.gpu

MATCH = 0.999


@functools.lru_cache(maxsize=None)
def _wl(name, **kw):
    from paper_2512_10520_b200 import workloads as w
    return getattr(w, name)(**dict(kw))


def _report(tag, c):
    print("%s: matched %.6f bit-exact %.6f max|dP|/P %.3g max|dr| %.3g" % (tag, c["matched"], c["bit_exact"], c["max_dp"], c["max_dr"]))


# ------------------------------------------------------------------------------------------- pieces
def test_philox_words_match_oracle(mt, oracle):
    b = mt.binding
    ctx = b.mt_create(0)
    try:
        for seed, id_base, step in ((1, 0, 0), (0x0123456789ABCDEF, 0xFFFFFFF0, 77), (2 ** 63 + 5, 2 ** 40 + 3, 4099)):
            n = 1000
            got = b.mt_debug_philox(ctx, seed, id_base, step, n).cpu().numpy().view(np.uint32)
            ctr = np.zeros((n, 4), np.uint32)
            ids = id_base + np.arange(n, dtype=np.uint64)
            ctr[:, 0] = (ids & 0xFFFFFFFF).astype(np.uint32)
            ctr[:, 1] = (ids >> np.uint64(32)).astype(np.uint32)
            ctr[:, 2] = step
            want = oracle.philox4x32_10(ctr, np.array([seed & 0xFFFFFFFF, seed >> 32], np.uint32))
            assert np.array_equal(got, want)
    finally:
        b.mt_destroy(ctx)


@pytest.mark.parametrize("shape", [(2, 5, 128, 64), (1, 3, 1024, 512), (3, 4, 7, 300)])
def test_alias_tables_and_draws_bit_exact(mt, oracle, shape):
    """mt_build_alias == the oracle's construction bit for bit; mt_debug_sample == oracle draw for the same words."""
    import torch
    from paper_2512_10520_b200.workloads import Histograms
    b = mt.binding
    M, nb, n_dp, n_th = shape
    rng = np.random.default_rng(sum(shape))
    cd = rng.gamma(0.4, 1.0, (M, nb, n_dp)).astype(np.float32)
    ct = rng.gamma(0.4, 1.0, (M, nb, n_th)).astype(np.float32)
    cd[rng.random(cd.shape) < 0.2] = 0.0
    cd[..., 0] += 1.0
    ct[0, 0, :] = 1.0                                    # a uniform table: every prob == 1
    h = Histograms(M, nb, n_dp, n_th, 1.0, 300.0, cd, ct, np.zeros((M, nb, 2), np.float32) + [-10.0, 0.01],
                   np.zeros((M, nb, 2), np.float32) + [-12.0, 0.02], np.full(M + 1, 0.02, np.float32))
    ctx = b.mt_create(0)
    try:
        b.mt_load_histograms(ctx, h)
        b.mt_build_alias(ctx)
        pd, ad, pt, at = b.mt_get_alias(ctx, h)
        opd, oad = oracle.build_alias(cd)
        opt, oat = oracle.build_alias(ct)
        assert np.array_equal(pd.view(np.uint32), opd.view(np.uint32)) and np.array_equal(ad, oad)
        assert np.array_equal(pt.view(np.uint32), opt.view(np.uint32)) and np.array_equal(at, oat)
        words = rng.integers(0, 2 ** 32, 200_000, dtype=np.uint64).astype(np.uint32)
        words[:4] = [0, 0xFFFFFFFF, 0x80000000, 1]
        dw = torch.from_numpy(words.view(np.int32)).cuda()
        for (m, i, which) in ((1, 0, 0), (M, nb - 1, 1), (1, 0, 1), (M, nb // 2, 0)):
            got = b.mt_debug_sample(ctx, m, i, which, dw).cpu().numpy().view(np.uint32)
            if which == 0:
                want = oracle.alias_draw(opd[m - 1, i], oad[m - 1, i], words)
            else:
                want = oracle.alias_draw(opt[m - 1, i], oat[m - 1, i], words)
            assert np.array_equal(got, want)
    finally:
        b.mt_destroy(ctx)


# ---------------------------------------------------------------------------------- configs, full size
def test_config0_toy_slab_full(mt, oracle):
    wl = _wl("config0")
    ref = oracle_transport(oracle, wl)
    # every muon exits after 51 steps near 48.5 GeV
    assert np.all(ref["flag"] == 2) and np.all(ref["steps"] == 51)
    for sched in (1, 2, 3):
        g = gpu_transport(mt, wl, sched=sched)
        c = compare(g, ref)
        _report("config0 sched %d" % sched, c)
        assert c["matched"] >= MATCH and c["bit_exact"] == 1.0
        assert g["counters"][0] == ref["steps"].sum() and g["counters"][2] == len(ref["flag"])


def test_config1_magnetised_block_full(mt, oracle):
    wl = _wl("config1")
    ref = oracle_transport(oracle, wl)
    assert set(np.unique(ref["flag"])) >= {2, 3}          # exits and lateral escapes both occur
    for sched, block in ((1, 128), (2, 256), (3, 64)):
        g = gpu_transport(mt, wl, sched=sched, block=block)
        c = compare(g, ref)
        _report("config1 sched %d" % sched, c)
        assert c["matched"] >= MATCH and c["bit_exact"] == 1.0
        assert all(p > 0.01 for p in ks_populations(g, ref).values())


def test_config2_multi_region_shield_full(mt, oracle):
    wl = _wl("config2")
    ref = oracle_transport(oracle, wl)
    g = gpu_transport(mt, wl)
    c = compare(g, ref)
    _report("config2", c)
    assert c["matched"] >= MATCH and c["bit_exact"] == 1.0
    assert all(p > 0.01 for p in ks_populations(g, ref).values())
    assert np.array_equal(g["counters"][1:5], np.bincount(ref["flag"], minlength=5)[1:5])


# ------------------------------------------------------------------- config 3: small grid, all muons
@pytest.mark.parametrize("sched", [1, 2, 3])
def test_config3_small_grid_elementwise(mt, oracle, sched):
    import torch
    from paper_2512_10520_b200 import workloads as w
    wl = w.config3(n=30_011, n_draws=100_000, n_cells=2, half_width_cells=40, device="cuda")
    wl.muons.mom[::7] *= np.float32(0.15)                 # a soft component (1.5 GeV and up) that ranges out in the iron
    ref = oracle_transport(oracle, wl)
    g = gpu_transport(mt, wl, sched=sched, slab=50 if sched == 3 else 0)
    c = compare(g, ref)
    _report("config3-small sched %d" % sched, c)
    assert len(np.unique(ref["flag"])) >= 3               # stopped, exited and escaped all occur
    assert c["matched"] >= MATCH and c["bit_exact"] == 1.0
    del wl
    torch.cuda.empty_cache()


def test_material_rides_with_the_field(mt, oracle):
    """The kernel reads the material from the packed field cell; exercise cell-boundary positions."""
    import torch
    from paper_2512_10520_b200 import workloads as w
    wl = w.config3(n=4096, n_draws=50_000, n_cells=1, half_width_cells=16, device="cuda")
    rng = np.random.default_rng(9)
    # starts exactly on cell faces and half-cells, in all three axes, heading in random directions
    k = rng.integers(-16, 16, (4096, 3))
    wl.muons.pos_q[:, 0] = (k[:, 0] * 0.01).astype(np.float32)
    wl.muons.pos_q[:, 1] = (k[:, 1] * 0.01 + 0.005 * (k[:, 2] % 2)).astype(np.float32)
    wl.muons.pos_q[:, 2] = (np.abs(k[:, 2]) * 0.01).astype(np.float32)
    d = rng.standard_normal((4096, 3))
    d[:, 2] = np.abs(d[:, 2]) + 0.2
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    wl.muons.mom[:, :3] = (d * rng.uniform(1.5, 40.0, (4096, 1))).astype(np.float32)
    ref = oracle_transport(oracle, wl)
    g = gpu_transport(mt, wl, sched=2)
    c = compare(g, ref)
    _report("cell faces", c)
    assert c["bit_exact"] == 1.0


# ------------------------------------------------------- config 3 at full size: sampled muons (ids)
def test_config3_full_size_sampled(mt, oracle):
    """BASELINE configs[3] as bench.py times it (10^7 muons, 200x200x3000 grid, default schedule); the oracle
    recomputes every 10th muon (10^6 of them: SURVEY.md §8(d)'s protocol when the oracle cannot do the whole batch in
    10 minutes) one by one from its id (muons are independent; RNG is keyed by id)."""
    import torch
    from paper_2512_10520_b200 import workloads as w
    b = mt.binding
    need_device_memory(12)
    wl = w.config3(device="cuda")
    n = len(wl.muons.pos_q)
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        g = gpu_transport(mt, wl, handle=h)
        assert g["counters"][1:5].sum() == n and g["counters"][0] == g["steps"].sum()
        sel = np.arange(0, n, 10)
        ref = oracle_transport(oracle, wl, sel=sel, ids=sel.astype(np.uint64))
        sub = {k: g[k][sel] for k in ("pos", "mom", "flag", "steps")}
        c = compare(sub, ref)
        _report("config3 full (every 10th)", c)
        assert c["matched"] >= MATCH and c["bit_exact"] == 1.0
        # properties that hold at any size
        assert np.all((g["flag"] >= 1) & (g["flag"] <= 4))
        P = np.linalg.norm(g["mom"].astype(np.float64), axis=1)
        assert np.all(P[g["flag"] == 1] < 1.0) and np.all(g["pos"][g["flag"] == 2][:, 2] >= 30.0)
        assert np.all(P <= np.linalg.norm(wl.muons.mom[:, :3].astype(np.float64), axis=1) * (1 + 1e-5))
    finally:
        h.close()
        del wl
        torch.cuda.empty_cache()


# --------------------------------------------- config 4: the three table shapes, batches with id_base
@pytest.mark.parametrize("shape", [(50, 128, 64), (100, 256, 128), (256, 1024, 512)])
def test_config4_table_shapes_and_batches(mt, oracle, shape):
    """BASELINE configs[4] on a reduced grid: every table shape of the sweep (pack32 and pack64 cells, shared-memory
    and L2 placement), two batches whose ids continue (id_base = batch * n), element by element."""
    import torch
    from paper_2512_10520_b200 import workloads as w
    b = mt.binding
    n = 20_011
    wl = w.config3(n=n, n_draws=30_000, n_cells=2, half_width_cells=40, device="cuda", table_shape=shape)
    T, G = oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom)
    placements = [b.MT_PLACE_AUTO, b.MT_PLACE_L2] + ([b.MT_PLACE_SMEM] if shape[0] <= 100 else [])
    for batch in (0, 1):
        mu = w.spectrum_muons(3, n, "square", batch=batch)
        mu.pos_q[:, :2] *= np.float32(0.4)
        mu.mom[::5] *= np.float32(0.2)
        wl.muons = mu
        ref = oracle_transport(oracle, wl, id_base=batch * n, tables=T, geom=G)
        for placement in placements:
            g = gpu_transport(mt, wl, placement=placement, id_base=batch * n)
            c = compare(g, ref)
            _report("config4 %dx%dx%d batch %d placement %d" % (shape + (batch, placement)), c)
            assert c["matched"] >= MATCH and c["bit_exact"] == 1.0
    del wl
    torch.cuda.empty_cache()


@pytest.mark.parametrize("shape,batch", [((256, 1024, 512), 3), ((100, 256, 128), 5), ((50, 128, 64), 7)])
def test_config4_full_size_sampled(mt, oracle, shape, batch):
    """BASELINE configs[4] as `bench.py --sweep` times it: the full 200x200x3000 grid, one 10^7-muon batch of the 10^8
    (generator batch and id_base = batch * 10^7 != 0), each of the three table shapes (8-byte cells, 9.4 MB; 4-byte
    cells from L2; fits shared memory); the oracle recomputes every 100th muon one by one from its id."""
    import torch
    from paper_2512_10520_b200 import workloads as w
    b = mt.binding
    need_device_memory(12)
    n = 10_000_000
    wl = w.config3(n=8, device="cuda", table_shape=shape, n_draws=200_000)
    wl.muons = w.spectrum_muons(3, n, "square", batch=batch)
    id_base = batch * n
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        g = gpu_transport(mt, wl, handle=h, id_base=id_base)
        assert b.mt_get_info(h.ctx, b.MT_INFO_LAST_SCHEDULE) == b.MT_SCHED_WAVEFRONT
        assert g["counters"][1:5].sum() == n and g["counters"][0] == g["steps"].sum()
        sel = np.arange(0, n, 100)
        ref = oracle_transport(oracle, wl, sel=sel, ids=(sel + id_base).astype(np.uint64))
        sub = {k: g[k][sel] for k in ("pos", "mom", "flag", "steps")}
        c = compare(sub, ref)
        _report("config4 full %dx%dx%d batch %d (every 100th)" % (shape + (batch,)), c)
        assert c["matched"] >= MATCH and c["bit_exact"] == 1.0
        assert np.all((g["flag"] >= 1) & (g["flag"] <= 4))
    finally:
        h.close()
        del wl
        torch.cuda.empty_cache()
