"""-m gpu: the SURVEY.md §8(f) variants and configs[4]'s largest launch IN THE LAUNCH CONFIGURATION bench.py times them in.

The element-by-element tests of test_gpu_variants.py / test_gpu_poly.py run 3e4-1e5 muons on an 80x80x750 grid with a
forced slab; the numbers in BASELINE.md / profiles come from other launch paths — 10^7 muons on the 200x200x3000 grid
(768-thread persistent CTAs, the AUTO slab of each field mode, L1-allocating grid loads for the per-stage kernels), 2^24
muons in one call, 10^6 muons through the polyhedra in two item-mode lanes.  Here each of those is launched as the bench
launches it (library defaults throughout), the context is asked which path it took, and the oracle recomputes a sample of
the muons one by one from their ids (every k-th muon when the oracle cannot do the batch), bit for bit.
"""
import copy

import numpy as np
import pytest

from gpu_util import compare, gpu_transport, need_device_memory, oracle_transport

pytestmark = pytest.mark.gpu
MATCH = 0.999


@pytest.fixture(scope="module")
def full3(workloads):
    """configs[3] at full size: the 200x200x3000 grids on the device (made once for this module) and 10^7 muons."""
    import torch
    need_device_memory(16)
    wl = workloads.config3(device="cuda", n_draws=200_000)
    yield wl
    wl.geom.material = wl.geom.field = None
    torch.cuda.empty_cache()


def _sampled(mt, oracle, wl, handle, stride, id_base, name):
    b = mt.binding
    n = len(wl.muons.pos_q)
    g = gpu_transport(mt, wl, handle=handle, id_base=id_base)
    assert g["counters"][1:5].sum() == n and g["counters"][0] == g["steps"].sum()
    assert np.all((g["flag"] >= 1) & (g["flag"] <= 4))
    sel = np.arange(0, n, stride)
    ref = oracle_transport(oracle, wl, sel=sel, ids=(sel + id_base).astype(np.uint64))
    c = compare({k: g[k][sel] for k in ("pos", "mom", "flag", "steps")}, ref)
    print("%s: every %dth of %d muons: matched %.5f bit-exact %.5f" % (name, stride, n, c["matched"], c["bit_exact"]))
    assert c["matched"] >= MATCH and c["bit_exact"] == 1.0, name
    facts = b.mt_get_info(handle.ctx, b.MT_INFO_LEAN_FACTS)
    return dict(schedule=b.mt_get_info(handle.ctx, b.MT_INFO_LAST_SCHEDULE), lanes=b.mt_get_info(handle.ctx, b.MT_INFO_LAST_LANES),
                lean=b.mt_get_info(handle.ctx, b.MT_INFO_LAST_LEAN), facts=facts)


@pytest.mark.parametrize("joint,field_mode,stride", [(True, 0, 100), (False, 1, 100), (False, 2, 200), (False, 3, 200),
                                                     (True, 2, 200)])
def test_config3_variants_full_size_sampled(mt, oracle, workloads, full3, joint, field_mode, stride):
    """`bench.py --joint` / `--field-mode 1|2|3` / both: 10^7 muons, library defaults."""
    b = mt.binding
    wl = copy.copy(full3)
    wl.geom = copy.copy(full3.geom)
    wl.geom.field_mode = field_mode
    if joint:
        wl.hist = workloads.shield_histograms(3, [1.0, 1.0, 10.0], 100, 256, 128, 200_000, joint=True)
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        took = _sampled(mt, oracle, wl, h, stride, 0, "config3 full joint=%d field_mode=%d" % (joint, field_mode))
        # the path the bench number comes from: one lane of z-slab passes, the LEAN kernel wherever its facts are proven
        assert took["schedule"] == b.MT_SCHED_WAVEFRONT and took["lanes"] == 1
        assert took["lean"] == int((took["facts"] & 3) == 3), took
    finally:
        h.close()


def test_config4_largest_launch_2_to_the_24(mt, oracle, workloads, full3):
    """BASELINE configs[4]: "muons-per-launch from 2^14 to 2^24" — the last point, 16 777 216 muons in ONE call (1.8 GB of
    wavefront scratch, ~1.8e10 muon-steps), with ids that do not start at 0; every 200th muon against the oracle."""
    b = mt.binding
    n = 1 << 24
    wl = copy.copy(full3)
    wl.muons = workloads.spectrum_muons(3, n, "square", batch=11)
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        took = _sampled(mt, oracle, wl, h, 200, 11 * 10_000_000, "config4 2^24 muons per launch")
        assert took["schedule"] == b.MT_SCHED_WAVEFRONT and took["lanes"] == 1
    finally:
        h.close()


def test_polyhedral_shield_at_bench_size(mt, oracle, workloads):
    """`bench.py --config 2 --poly --muons 1000000`: 10^6 muons through the tapered-magnet polyhedra — z-slab passes in two
    item-mode lanes (the launch path of the 2p number); every 4th muon against the oracle (its block scan is linear)."""
    b = mt.binding
    wl = workloads.config2p(n=1_000_000, n_draws=200_000)
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        took = _sampled(mt, oracle, wl, h, 4, 0, "config2p at 10^6")
        assert took["schedule"] == b.MT_SCHED_WAVEFRONT and took["lanes"] == 2
    finally:
        h.close()


@pytest.mark.parametrize("half_width_cells,n_cells", [(50, 8), (200, 4)])
def test_other_voxel_grids_under_the_default_slab(mt, oracle, workloads, half_width_cells, n_cells):
    """The AUTO slab and CTA shape were tuned on configs[3]'s 200x200x3000 grid (1.3 MB per padded layer).  Grids with a
    quarter and four times that layer — 100x100x3000 and 400x400x1500, where 96 layers are 32 MB and 500 MB against 126 MB
    of L2 — go through the same full-batch launch path (2.5e6 muons: one lane, 96-cell slabs); every 50th muon against the
    oracle.  (profiles/r3_slab_grids.md has the slab sweep on the three grids: AUTO is within 0.8 % of the best fixed slab.)"""
    import torch
    b = mt.binding
    need_device_memory(24)
    n = 2_500_000
    wl = workloads.config3(n=n, n_draws=200_000, n_cells=n_cells, half_width_cells=half_width_cells, device="cuda")
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        took = _sampled(mt, oracle, wl, h, 50, 3 * n, "voxel grid %dx%dx%d" % (wl.geom.nx, wl.geom.ny, wl.geom.nz))
        assert took["schedule"] == b.MT_SCHED_WAVEFRONT and took["lanes"] == 1
    finally:
        h.close()
        wl.geom.material = wl.geom.field = None
        del wl
        torch.cuda.empty_cache()
