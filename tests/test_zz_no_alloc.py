"""-m gpu: mt_transport_static_scratch, the transport call for callers that cannot allocate device memory.

Some users of this library run where a cudaMalloc is not an option once they are going: all of the GPU's memory already
belongs to a framework's pool or to a budget fixed at start-up, or they sit in a latency-bound loop that cannot afford the
device-wide stall of cudaMalloc / cudaFree.  mt_transport allocates (its scratch grows with the largest batch seen, its
lanes need streams and events), so they get an entry point of their own whose scratch is a fixed array inside the library's
image; include/muon_transport.h states the contract.  What is checked here:

  * its outputs equal mt_transport's bit for bit (the tolerance the launch-independence tests use: a schedule or a launch
    shape never changes a result), under each schedule, on calls made back to back on one stream — the array still holds
    the previous call's counters, histogram and parked muons, so a missing clear shows up in the second call;
  * a batch above MT_STATIC_SCRATCH_MAX_MUONS is refused with a message that names the limit, and nothing is written.

This file sorts last on purpose (pytest -x stops at the first failure; the new entry point must not hide the rest), and it
passes on its own in a fresh process, where its first call is also the library's first use of the array on the device.
"""
import numpy as np
import pytest

from gpu_util import unpack

pytestmark = pytest.mark.gpu


def _as_numpy(out, exit_capacity):
    res = unpack(out["pos_flag"].cpu().numpy(), out["mom_steps"].cpu().numpy())
    res["counters"] = out["counters"].cpu().numpy()
    if exit_capacity:
        res["exit_count"] = int(out["exit_count"].cpu().numpy()[0])
        rec = out["exit_rec"].cpu().numpy()[:min(res["exit_count"], exit_capacity)].view(np.uint32)
        res["exit_rec"] = rec[np.argsort(rec[:, 3], kind="stable")]       # (the list's order is whoever came first)
    return res


def _existing_path(h, dq, dm, seed, id_base, exit_capacity):
    import torch
    out = h.transport(dq, dm, seed, id_base=id_base, exit_capacity=exit_capacity)
    torch.cuda.synchronize()
    return _as_numpy(out, exit_capacity)


def _static_scratch(h, dq, dm, seed, id_base, exit_capacity, out=None):
    """Every buffer is the caller's; the binding allocates nothing."""
    import torch
    n = dq.shape[0]
    if out is None:
        out = {"pos_flag": torch.empty((n, 4), dtype=torch.float32, device="cuda"),
               "mom_steps": torch.empty((n, 4), dtype=torch.float32, device="cuda"),
               "counters": torch.zeros(8, dtype=torch.int64, device="cuda")}
        if exit_capacity:
            out["exit_rec"] = torch.zeros((exit_capacity, 8), dtype=torch.float32, device="cuda")
            out["exit_count"] = torch.zeros(1, dtype=torch.int32, device="cuda")
    return h.transport_static_scratch(dq, dm, seed, out, id_base=id_base)


def _assert_same(a, b, what):
    for k in ("pos", "mom"):
        assert np.array_equal(a[k].view(np.uint32), b[k].view(np.uint32)), (what, k)
    for k in ("flag", "steps", "counters"):
        assert np.array_equal(a[k], b[k]), (what, k)
    if "exit_rec" in b:
        assert a["exit_count"] == b["exit_count"], what
        assert np.array_equal(a["exit_rec"], b["exit_rec"]), (what, "exit_rec")


def _back_to_back(mt, wl, settings, exit_capacity):
    """Three calls in a row on one stream — a large batch, a smaller one with other ids (so the array holds MORE leftovers
    than the call uses), the large one again — each checked against mt_transport on the same inputs."""
    import torch
    b = mt.binding
    n = len(wl.muons.pos_q)
    dq_all = torch.from_numpy(np.ascontiguousarray(wl.muons.pos_q)).cuda()
    dm_all = torch.from_numpy(np.ascontiguousarray(wl.muons.mom)).cuda()
    calls = [(slice(0, n), 0), (slice(n // 3, n // 3 + n // 4 + 5), 2 ** 33 + n // 3), (slice(0, n), 0)]
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        for opts in settings:
            for name, value in {**dict(sched=0, block=0, slab=0, sort_every=0), **opts}.items():
                h.set_option({"sched": b.MT_OPT_SCHEDULE, "block": b.MT_OPT_BLOCK_THREADS, "slab": b.MT_OPT_SLAB_CELLS,
                              "sort_every": b.MT_OPT_SORT_EVERY}[name], value)
            want = [_existing_path(h, dq_all[s].contiguous(), dm_all[s].contiguous(), wl.seed, base, exit_capacity)
                    for s, base in calls]
            outs = [_static_scratch(h, dq_all[s].contiguous(), dm_all[s].contiguous(), wl.seed, base, exit_capacity)
                    for s, base in calls]                         # enqueued back to back, nothing in between
            assert b.mt_get_info(h.ctx, b.MT_INFO_LAST_LANES) == 1
            if opts.get("sched"):
                assert b.mt_get_info(h.ctx, b.MT_INFO_LAST_SCHEDULE) == opts["sched"]
            torch.cuda.synchronize()
            for k, (got, ref) in enumerate(zip(outs, want)):
                _assert_same(_as_numpy(got, exit_capacity), ref, (opts, "call %d" % k))
            errors = b.mt_get_info(h.ctx, b.MT_INFO_CHECK_ERRORS)          # (the bounds-checked build, if that is what is loaded)
            assert errors in (0, -1), errors
    finally:
        h.close()


def test_static_scratch_equals_mt_transport_on_the_field_map(mt, workloads):
    """Voxel grid + trilinear field (configs[3], shrunk): AUTO takes z-slab passes; thin slabs give ~75 passes, each
    with its own counter, parked records that alternate between the two buffers, and a sort between passes."""
    wl = workloads.config3(n=24_001, n_draws=50_000, n_cells=2, half_width_cells=40, device="cuda")
    _back_to_back(mt, wl, [dict(), dict(sched=3, slab=10), dict(sched=3, slab=37, sort_every=3, block=96), dict(sched=2),
                           dict(sched=1)], exit_capacity=30_000)


def test_static_scratch_equals_mt_transport_in_regions(mt, workloads):
    """Box regions with a uniform field (configs[1]): AUTO takes the persistent REFILL kernel, whose scratch is the
    counter idle lanes draw new muons from — left at its final value by the call before."""
    wl = workloads.config1(n=20_000, n_draws=100_000)
    _back_to_back(mt, wl, [dict(), dict(sched=3, slab=25)], exit_capacity=0)


def test_static_scratch_refuses_what_does_not_fit(mt, workloads):
    import torch
    b = mt.binding
    assert b.MT_STATIC_SCRATCH_MAX_MUONS == 65536
    wl = workloads.config1(n=64, n_draws=50_000)
    h = b.MuonTransport(0).setup(wl.hist, wl.geom)
    try:
        n = b.MT_STATIC_SCRATCH_MAX_MUONS + 1
        dq = torch.from_numpy(np.ascontiguousarray(wl.muons.pos_q)).cuda().repeat(n // 64 + 1, 1)[:n].contiguous()
        dm = torch.from_numpy(np.ascontiguousarray(wl.muons.mom)).cuda().repeat(n // 64 + 1, 1)[:n].contiguous()
        out = {"pos_flag": torch.full((n, 4), -7.0, device="cuda"), "mom_steps": torch.full((n, 4), -7.0, device="cuda")}
        for sched in (0, 1, 2, 3):                      # the limit is the entry point's, whatever the schedule would need
            h.set_option(b.MT_OPT_SCHEDULE, sched)
            with pytest.raises(b.MtError) as err:
                h.transport_static_scratch(dq, dm, wl.seed, out)
            assert err.value.code == b.MT_ERR_UNSUPPORTED
            assert "65536" in str(err.value) and "mt_transport" in str(err.value)
        torch.cuda.synchronize()
        assert bool((out["pos_flag"] == -7.0).all()) and bool((out["mom_steps"] == -7.0).all())
        # exactly the maximum is served, and an empty call is a no-op
        h.set_option(b.MT_OPT_SCHEDULE, 3)
        n = b.MT_STATIC_SCRATCH_MAX_MUONS
        got = _static_scratch(h, dq[:n].contiguous(), dm[:n].contiguous(), wl.seed, 5, 0)
        ref = _existing_path(h, dq[:n].contiguous(), dm[:n].contiguous(), wl.seed, 5, 0)
        torch.cuda.synchronize()
        _assert_same(_as_numpy(got, 0), ref, "n = maximum")
        empty = torch.zeros((0, 4), device="cuda")
        h.transport_static_scratch(empty, empty, 1, {"pos_flag": empty.clone(), "mom_steps": empty.clone()})
    finally:
        h.close()
