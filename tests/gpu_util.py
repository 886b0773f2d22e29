"""Helpers shared by the -m gpu parity tests: run a workload through the C ABI and through the oracle."""
import numpy as np


def need_device_memory(gib):
    """The full-size parity tests need `gib` GiB free.  On a small development GPU they skip; on a B200-class device
    (>= 150 GiB in all) too little free memory is a FAILURE: there the headline configurations must be checked, and a
    silent skip would turn their parity into "untested"."""
    import pytest
    import torch
    free, total = torch.cuda.mem_get_info()
    if free >= gib * 2 ** 30:
        return
    msg = "needs %d GiB of device memory, %.1f GiB free of %.1f" % (gib, free / 2 ** 30, total / 2 ** 30)
    if total >= 150 * 2 ** 30:
        pytest.fail(msg + ": on this device the full-size parity tests must run")
    pytest.skip(msg)


def gpu_transport(mt, wl, sched=0, block=0, placement=0, id_base=0, exit_capacity=0, min_idle=0, slab=0,
                  sel=None, handle=None, lanes=0, pass_mode=0, lane_prio=0, sort_every=0):
    """Run workload `wl` on cuda:0 through the binding; returns numpy dict (pos, mom, flag, steps, ...)."""
    import torch
    b = mt.binding
    own = handle is None
    h = handle or b.MuonTransport(0).setup(wl.hist, wl.geom, placement)
    try:
        h.set_option(b.MT_OPT_SCHEDULE, sched).set_option(b.MT_OPT_BLOCK_THREADS, block)
        h.set_option(b.MT_OPT_REFILL_MIN_IDLE, min_idle).set_option(b.MT_OPT_SLAB_CELLS, slab)
        h.set_option(b.MT_OPT_LANES, lanes).set_option(b.MT_OPT_PASS_MODE, pass_mode).set_option(b.MT_OPT_LANE_PRIORITY, lane_prio)
        h.set_option(b.MT_OPT_SORT_EVERY, sort_every)
        pos_q, mom = wl.muons.pos_q, wl.muons.mom
        if sel is not None:
            pos_q, mom = pos_q[sel], mom[sel]
        dq = torch.from_numpy(np.ascontiguousarray(pos_q)).cuda()
        dm = torch.from_numpy(np.ascontiguousarray(mom)).cuda()
        out = h.transport(dq, dm, wl.seed, id_base=id_base, exit_capacity=exit_capacity)
        torch.cuda.synchronize()
        res = unpack(out["pos_flag"].cpu().numpy(), out["mom_steps"].cpu().numpy())
        res["counters"] = out["counters"].cpu().numpy()
        if exit_capacity:
            res["exit_count"] = int(out["exit_count"].cpu().numpy()[0])
            res["exit_rec"] = out["exit_rec"].cpu().numpy()
        # checked build (MUON_TRANSPORT_LIB=...libmuon_transport_checked.so): no index left its array
        errors = b.mt_get_info(h.ctx, b.MT_INFO_CHECK_ERRORS)
        assert errors in (0, -1), "bounds violations: %d, highest code %d" % (errors & 0xFFFFFFFF, errors >> 32)
        return res
    finally:
        if own:
            h.close()


def unpack(pos_flag, mom_steps):
    return dict(pos=pos_flag[:, :3].copy(), mom=mom_steps[:, :3].copy(),
                flag=pos_flag[:, 3].copy().view(np.int32), steps=mom_steps[:, 3].copy().view(np.int32))


def oracle_transport(oracle, wl, sel=None, id_base=0, ids=None, tables=None, geom=None):
    pos_q, mom = wl.muons.pos_q, wl.muons.mom
    if sel is not None:
        pos_q, mom = pos_q[sel], mom[sel]
    T = tables or oracle.OracleTables(wl.hist)
    G = geom or oracle.OracleGeometry(wl.geom)
    return oracle.transport(T, G, pos_q, mom, wl.seed, id_base=id_base, ids=ids, threads=oracle.max_threads())


def compare(gpu, ref, tol_p=1e-5, tol_r=1e-5):
    """north_star's per-muon criteria.  Returns dict of fractions and the mask of matched muons."""
    same_meta = (gpu["flag"] == ref["flag"]) & (gpu["steps"] == ref["steps"])
    Pg = np.linalg.norm(gpu["mom"].astype(np.float64), axis=1)
    Pr = np.linalg.norm(ref["mom"].astype(np.float64), axis=1)
    dp = np.abs(Pg - Pr) / np.maximum(Pr, 1e-30)
    dr = np.linalg.norm(gpu["pos"].astype(np.float64) - ref["pos"].astype(np.float64), axis=1)
    ok = same_meta & (dp <= tol_p) & (dr <= tol_r)
    bit = same_meta & np.all(gpu["pos"].view(np.uint32) == ref["pos"].view(np.uint32), axis=1) \
        & np.all(gpu["mom"].view(np.uint32) == ref["mom"].view(np.uint32), axis=1)
    n = max(len(ok), 1)
    return dict(matched=ok.sum() / n, bit_exact=bit.sum() / n, mask=ok, max_dp=float(dp.max(initial=0)),
                max_dr=float(dr.max(initial=0)))


def ks_populations(gpu, ref):
    """two-sample KS p-values on final p, theta, x, y (north_star)"""
    from scipy import stats
    out = {}
    for name, f in (("p", lambda d: np.linalg.norm(d["mom"].astype(np.float64), axis=1)),
                    ("theta", lambda d: np.arccos(np.clip(d["mom"][:, 2].astype(np.float64) /
                                                          np.maximum(np.linalg.norm(d["mom"].astype(np.float64), axis=1), 1e-30), -1, 1))),
                    ("x", lambda d: d["pos"][:, 0].astype(np.float64)),
                    ("y", lambda d: d["pos"][:, 1].astype(np.float64))):
        out[name] = stats.ks_2samp(f(gpu), f(ref)).pvalue
    return out
