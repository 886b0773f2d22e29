"""Target program for memory checking (not a pytest file):

    MUON_TRANSPORT_LIB=paper_2512_10520_b200/libmuon_transport_checked.so python tests/sanitize_target.py --checked
    compute-sanitizer --tool memcheck  python tests/sanitize_target.py [--quick]      (where the tool is available)
    compute-sanitizer --tool racecheck python tests/sanitize_target.py [--quick]

--checked: the library is the bounds-checked build (paper_2512_10520_b200/build.py --checked); every case must finish
with zero violations, and a self-test that hands the kernels a wrong table size must make the checks fire.

Small transports through every schedule (STATIC, REFILL, WAVEFRONT: park / index-sort path with its per-key atomics,
single-CTA scan and alternating record buffers), both table placements (L2 gathers and the shared-memory staged copy),
the three geometries and the host-buffer call, each checked bit for bit against the oracle so that a sanitizer-clean
run is also a correct one.  Sizes are tiny: the tools slow kernels down by one to two orders of magnitude.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def main():
    import torch
    import oracle
    import paper_2512_10520_b200 as mt
    from paper_2512_10520_b200 import workloads as w
    from gpu_util import compare, gpu_transport, oracle_transport, unpack
    b = mt.binding
    quick = "--quick" in sys.argv
    n = 600 if quick else 3000
    cases = []
    wl3 = w.config3(n=n, n_draws=20_000, n_cells=1, half_width_cells=16, device="cuda")
    wl3.muons.mom[::3] *= np.float32(0.3)
    ref3 = oracle_transport(oracle, wl3)
    for sched in (1, 2, 3):
        for placement in (b.MT_PLACE_L2, b.MT_PLACE_SMEM):
            cases.append(("voxel sched %d placement %d" % (sched, placement), wl3, ref3,
                          dict(sched=sched, placement=placement, slab=40 if sched == 3 else 0, exit_capacity=n)))
    wl2 = w.config2(n=n, n_draws=20_000, n_cells=1)
    ref2 = oracle_transport(oracle, wl2)
    for sched in (2, 3):
        cases.append(("regions sched %d" % sched, wl2, ref2, dict(sched=sched, placement=b.MT_PLACE_SMEM, exit_capacity=16)))
    wlp = w.config2p(n=n, n_draws=20_000, n_cells=1)
    refp = oracle_transport(oracle, wlp)
    for sched in (2, 3):
        cases.append(("polyhedra sched %d" % sched, wlp, refp, dict(sched=sched)))
    if not quick:
        wlj = w.config3(n=n, n_draws=20_000, n_cells=1, half_width_cells=16, device="cuda", joint=True,
                        table_shape=(20, 32, 16), field_mode=3)
        cases.append(("voxel joint, nearest per stage", wlj, oracle_transport(oracle, wlj), dict(sched=3, slab=50)))
    for name, wl, ref, kw in cases:
        g = gpu_transport(mt, wl, **kw)
        c = compare(g, ref)
        print("%-40s bit-exact %.4f  steps %d" % (name, c["bit_exact"], int(g["counters"][0])), flush=True)
        assert c["bit_exact"] == 1.0, name
    h = b.MuonTransport(0).setup(wl3.hist, wl3.geom)
    out = h.transport_host(wl3.muons.pos_q, wl3.muons.mom, wl3.seed, exit_capacity=64)
    assert compare(unpack(out["pos_flag"], out["mom_steps"]), ref3)["bit_exact"] == 1.0
    h.set_option(b.MT_OPT_LANES, 3)
    out = h.transport_host(wl3.muons.pos_q, wl3.muons.mom, wl3.seed, exit_capacity=64)
    assert compare(unpack(out["pos_flag"], out["mom_steps"]), ref3)["bit_exact"] == 1.0
    if "--checked" in sys.argv:
        assert b.mt_get_info(h.ctx, b.MT_INFO_CHECK_ERRORS) == 0, "this is not the checked build, or a check fired"
        # the checks are alive: with a table size of one cell nearly every alias draw is out of bounds (and is counted,
        # not dereferenced)
        h.set_option(b.MT_OPT_CHECK_SELFTEST, 1)
        h.transport_host(wl3.muons.pos_q, wl3.muons.mom, wl3.seed)
        errors = b.mt_get_info(h.ctx, b.MT_INFO_CHECK_ERRORS)
        assert (errors & 0xFFFFFFFF) > 1000 and (errors >> 32) == 6, errors            # MT_CHK_TABLE
        print("checked build: 0 violations in every case; self-test fired %d times (code %d)" % (errors & 0xFFFFFFFF, errors >> 32))
    h.close()
    torch.cuda.synchronize()
    print("sanitize_target: all cases bit-exact against the oracle")


if __name__ == "__main__":
    main()
