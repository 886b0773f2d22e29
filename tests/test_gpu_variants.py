"""-m gpu: the SURVEY.md §8(f) variants of the CUDA path against the oracle, element by element — the paper's joint 2D
histogram mode and the nearest-neighbour / per-stage field lookups (§3.11).  Same bar as
test_gpu_parity.py: north_star's tolerances and, because both sides evaluate one float32 contract, 100 % bit-exact."""
import numpy as np
import pytest

from gpu_util import compare, gpu_transport, ks_populations, oracle_transport

pytestmark = pytest.mark.gpu

MATCH = 0.999


def _check(tag, g, ref, ks=False):
    c = compare(g, ref)
    print("%s: matched %.6f bit-exact %.6f max|dP|/P %.3g max|dr| %.3g" % (tag, c["matched"], c["bit_exact"], c["max_dp"], c["max_dr"]))
    assert c["matched"] >= MATCH and c["bit_exact"] == 1.0
    if ks:
        assert all(p > 0.01 for p in ks_populations(g, ref).values())


@pytest.mark.parametrize("shape", [(1, 3, 16, 8), (2, 2, 128, 64), (1, 2, 300, 7), (1, 1, 1024, 512), (1, 2, 5, 1)])
def test_joint_tables_and_two_word_draws_bit_exact(mt, oracle, shape):
    import torch
    from paper_2512_10520_b200.workloads import Histograms
    b = mt.binding
    M, nb, n_a, n_b = shape
    rng = np.random.default_rng(sum(shape))
    counts = rng.gamma(0.3, 1.0, (M, nb, n_a, n_b)).astype(np.float32)
    counts[rng.random(counts.shape) < 0.3] = 0.0
    counts[..., 0, 0] += 1.0
    h = Histograms(M, nb, n_a, n_b, 1.0, 300.0, counts, None, np.zeros((M, nb, 2), np.float32) + [-10.0, 0.01],
                   np.zeros((M, nb, 2), np.float32) + [-12.0, 0.02], np.full(M + 1, 0.02, np.float32), joint=True)
    ctx = b.mt_create(0)
    try:
        b.mt_load_histograms(ctx, h)
        b.mt_build_alias(ctx)
        prob, alias, _, _ = b.mt_get_alias(ctx, h)
        oprob, oalias = oracle.build_alias(counts.reshape(M, nb, n_a * n_b))
        assert np.array_equal(prob.view(np.uint32), oprob.view(np.uint32)) and np.array_equal(alias, oalias)
        n = 100_000
        ws = rng.integers(0, 2 ** 32, n, dtype=np.uint64).astype(np.uint32)
        wa = rng.integers(0, 2 ** 32, n, dtype=np.uint64).astype(np.uint32)
        ws[:4] = [0, 0xFFFFFFFF, 0x80000000, 1]
        wa[:4] = [0xFFFFFFFF, 0, 0x000000FF, 0x00000100]
        dw = torch.from_numpy(np.concatenate([ws, wa]).view(np.int32)).cuda()
        for (m, i) in ((1, 0), (M, nb - 1)):
            got = b.mt_debug_sample(ctx, m, i, 0, dw, joint=True).cpu().numpy().view(np.uint32)
            assert np.array_equal(got, oracle.alias_draw2(oprob[m - 1, i], oalias[m - 1, i], ws, wa))
    finally:
        b.mt_destroy(ctx)


def test_joint_mode_configs_0_1_2(mt, oracle):
    from paper_2512_10520_b200 import workloads as w
    wl = w.config0(n_draws=200_000, joint=True)
    ref = oracle_transport(oracle, wl)
    assert np.all(ref["flag"] == 2) and np.all(ref["steps"] == 51)
    for sched in (1, 2, 3):
        _check("joint config0 sched %d" % sched, gpu_transport(mt, wl, sched=sched), ref)
    wl = w.config1(n_draws=200_000, joint=True)
    ref = oracle_transport(oracle, wl)
    for sched in (1, 2, 3):
        _check("joint config1 sched %d" % sched, gpu_transport(mt, wl, sched=sched), ref, ks=True)
    wl = w.config2(n=200_000, n_draws=60_000, joint=True, table_shape=(100, 64, 32))
    ref = oracle_transport(oracle, wl)
    assert len(np.unique(ref["flag"])) >= 3
    _check("joint config2", gpu_transport(mt, wl), ref, ks=True)


@pytest.mark.parametrize("joint,field_mode", [(True, 0), (False, 1), (False, 2), (False, 3), (True, 3)])
def test_config3_small_grid_variants(mt, oracle, joint, field_mode):
    import torch
    from paper_2512_10520_b200 import workloads as w
    shape = (100, 64, 32) if joint else (100, 256, 128)
    wl = w.config3(n=30_011, n_draws=60_000, n_cells=2, half_width_cells=40, device="cuda", joint=joint,
                   field_mode=field_mode, table_shape=shape)
    wl.muons.mom[::7] *= np.float32(0.15)
    ref = oracle_transport(oracle, wl)
    assert len(np.unique(ref["flag"])) >= 3
    for sched in (1, 2, 3):
        g = gpu_transport(mt, wl, sched=sched, slab=50 if sched == 3 else 0)
        _check("config3-small joint=%d field=%d sched %d" % (joint, field_mode, sched), g, ref)
    del wl
    torch.cuda.empty_cache()


def test_field_variants_change_the_answer_as_they_should(mt, oracle):
    """The variants are not no-ops: on the perturbed field map nearest and per-stage lookups move the final states,
    by amounts consistent with a 0.1 T perturbation over 1-cm cells."""
    import torch
    from paper_2512_10520_b200 import workloads as w
    base = w.config3(n=5000, n_draws=40_000, n_cells=1, half_width_cells=40, device="cuda")
    outs = {}
    for fm in (0, 1, 2):
        base.geom.field_mode = fm
        outs[fm] = gpu_transport(mt, base)
    same = outs[0]["flag"] == outs[1]["flag"]
    d1 = np.linalg.norm(outs[1]["pos"][same] - outs[0]["pos"][same], axis=1)
    d2 = np.linalg.norm(outs[2]["pos"][same] - outs[0]["pos"][same], axis=1)
    assert 0 < np.median(d1) < 0.05 and 0 < np.median(d2) < 0.05
    del base
    torch.cuda.empty_cache()


def test_per_stage_field_in_region_mode(mt, oracle):
    from paper_2512_10520_b200 import workloads as w
    wl = w.config2(n=100_000, n_draws=60_000)
    wl.geom.field_mode = 2
    ref = oracle_transport(oracle, wl)
    for sched in (2, 3):
        _check("config2 per-stage sched %d" % sched, gpu_transport(mt, wl, sched=sched), ref)
    wl.geom.field_mode = 0
    frozen = oracle_transport(oracle, wl)
    assert not np.array_equal(frozen["pos"], ref["pos"])          # region boundaries are seen by the stages


def test_variant_error_behaviour(mt):
    from paper_2512_10520_b200 import workloads as w
    b = mt.binding
    wl = w.config0(n=16, n_draws=20_000)
    h = b.MuonTransport(0)
    try:
        wl.geom.field_mode = 1                                    # nearest needs a voxel geometry
        with pytest.raises(b.MtError) as e:
            h.setup(wl.hist, wl.geom)
        assert e.value.code == b.MT_ERR_INVALID_ARG
        wl.geom.field_mode = 7
        with pytest.raises(b.MtError):
            h.setup(wl.hist, wl.geom)
        from paper_2512_10520_b200.workloads import Histograms
        big = Histograms(1, 1, 65536, 512, 1.0, 300.0, np.ones((1, 1, 2, 2), np.float32), None, np.zeros((1, 1, 2), np.float32),
                         np.zeros((1, 1, 2), np.float32), np.full(2, 0.02, np.float32), joint=True)
        d = b.mt_hist_desc(1, 1, 1.0, 300.0, 65536, 512, big.counts_dp.ctypes.data, None, big.axis_dp.ctypes.data,
                           big.axis_th.ctypes.data, big.step_m.ctypes.data, b.MT_HIST_JOINT)
        import ctypes
        assert b.lib().mt_load_histograms(h.ctx, ctypes.byref(d)) == b.MT_ERR_UNSUPPORTED      # 2^25 cells
    finally:
        h.close()
