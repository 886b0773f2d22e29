"""ctypes binding of libmuon_transport.so: the same calls as include/muon_transport.h, argument marshalling
only.  Every step of the transport path runs in the CUDA kernels behind the C ABI; there is no Python or CPU
fallback — a missing library or a missing CUDA device raises.  PyTorch supplies device memory and streams.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
# MUON_TRANSPORT_LIB: an alternative build of the same sources (build.py --checked: bounds-checked kernels) for tests
LIB_PATH = os.environ.get("MUON_TRANSPORT_LIB") or os.path.join(HERE, "libmuon_transport.so")

MT_OK = 0
MT_ERR_INVALID_ARG, MT_ERR_STATE, MT_ERR_EMPTY_HIST, MT_ERR_UNSUPPORTED, MT_ERR_CUDA, MT_ERR_NOMEM = -1, -2, -3, -4, -5, -6
MT_FLAG_STOPPED, MT_FLAG_EXITED, MT_FLAG_ESCAPED, MT_FLAG_MAXSTEPS = 1, 2, 3, 4
MT_GEOM_REGIONS, MT_GEOM_VOXEL, MT_GEOM_POLY = 0, 1, 2
MT_PLACE_AUTO, MT_PLACE_SMEM, MT_PLACE_L2 = 0, 1, 2
MT_SCHED_AUTO, MT_SCHED_STATIC, MT_SCHED_REFILL, MT_SCHED_WAVEFRONT = 0, 1, 2, 3
MT_OPT_SCHEDULE, MT_OPT_BLOCK_THREADS, MT_OPT_BLOCKS_PER_SM, MT_OPT_SLAB_CELLS, MT_OPT_REFILL_MIN_IDLE = 1, 2, 3, 4, 5
MT_OPT_KEY_LOOKAHEAD, MT_OPT_HASH_NXY, MT_OPT_HASH_NZ, MT_OPT_NO_LEAN, MT_OPT_LANES, MT_OPT_CHECK_SELFTEST = 6, 7, 8, 9, 10, 11
MT_OPT_PASS_MODE, MT_OPT_LANE_PRIORITY, MT_OPT_SORT_EVERY = 12, 13, 14
MT_HIST_MARGINAL, MT_HIST_JOINT = 0, 1
MT_EXIT_AT_BREAK, MT_EXIT_PROJECT = 0, 1
MT_INFO_LEAN_FACTS, MT_INFO_LAST_LEAN, MT_INFO_LAST_SCHEDULE, MT_INFO_LAST_LANES, MT_INFO_CHECK_ERRORS = 1, 2, 3, 4, 5
MT_FIELD_TRILINEAR, MT_FIELD_NEAREST, MT_FIELD_PER_STAGE = 0, 1, 2
MT_STATIC_SCRATCH_MAX_MUONS, MT_STATIC_SCRATCH_BYTES = 65536, 9 * 1024 * 1024

# every symbol include/muon_transport.h declares (tests check that the library exports each one)
SYMBOLS = ["mt_strerror", "mt_last_error", "mt_create", "mt_destroy", "mt_set_option", "mt_load_histograms",
           "mt_build_alias", "mt_get_alias", "mt_set_geometry", "mt_transport", "mt_transport_host",
           "mt_transport_static_scratch", "mt_launch_count", "mt_get_info", "mt_debug_sample", "mt_debug_philox", "mt_debug_lookup"]
# include/muon_probes.h: the measurement probes, in a library of their own (libmuon_probes.so) that the product never loads
PROBES_LIB_PATH = os.path.join(HERE, "libmuon_probes.so")
PROBE_SYMBOLS = ["mt_measure_peaks", "mt_probe_field_paths"]


class mt_hist_desc(C.Structure):
    _fields_ = [("n_materials", C.c_int32), ("n_pbins", C.c_int32), ("p_lo", C.c_float), ("p_hi", C.c_float),
                ("n_dp", C.c_int32), ("n_th", C.c_int32),
                ("counts_dp", C.c_void_p), ("counts_th", C.c_void_p), ("axis_dp", C.c_void_p),
                ("axis_th", C.c_void_p), ("step_m", C.c_void_p), ("hist_mode", C.c_int32)]


class mt_region(C.Structure):
    _fields_ = [("z_lo", C.c_float), ("z_hi", C.c_float), ("x_lo", C.c_float), ("x_hi", C.c_float),
                ("y_lo", C.c_float), ("y_hi", C.c_float), ("material", C.c_int32),
                ("bx", C.c_float), ("by", C.c_float), ("bz", C.c_float)]


class mt_poly_block(C.Structure):
    _fields_ = [("z_lo", C.c_float), ("z_hi", C.c_float), ("xy_lo", C.c_float * 2 * 4), ("xy_hi", C.c_float * 2 * 4),
                ("material", C.c_int32), ("bx", C.c_float), ("by", C.c_float), ("bz", C.c_float)]


class mt_geometry(C.Structure):
    _fields_ = [("mode", C.c_int32),
                ("x_min", C.c_float), ("x_max", C.c_float), ("y_min", C.c_float), ("y_max", C.c_float),
                ("z_min", C.c_float), ("z_exit", C.c_float),
                ("p_min", C.c_float), ("max_steps", C.c_int32), ("world_material", C.c_int32),
                ("n_regions", C.c_int32), ("regions", C.c_void_p),
                ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("ox", C.c_float), ("oy", C.c_float), ("oz", C.c_float), ("cell", C.c_float),
                ("d_material", C.c_void_p), ("d_field", C.c_void_p), ("field_mode", C.c_int32),
                ("n_blocks", C.c_int32), ("blocks", C.c_void_p), ("exit_mode", C.c_int32)]


class mt_peaks(C.Structure):
    _fields_ = [("sm_count", C.c_int32), ("sm_clock_mhz_nominal", C.c_double),
                ("ffma_thread_ops_per_s", C.c_double), ("ffma_warp_instr_per_s_per_smsp", C.c_double),
                ("lop3_thread_ops_per_s", C.c_double), ("imad_thread_ops_per_s", C.c_double),
                ("mulhi_thread_ops_per_s", C.c_double), ("mufu_thread_ops_per_s", C.c_double),
                ("gather_l1_bytes_per_s", C.c_double), ("gather_675k_bytes_per_s", C.c_double),
                ("gather_64m_bytes_per_s", C.c_double), ("gather_1400m_bytes_per_s", C.c_double),
                ("mix_ffma8_lop3_4_thread_ops_per_s", C.c_double), ("mix_ffma8_imad4_thread_ops_per_s", C.c_double),
                ("mix_ffma8_mulwide2_thread_ops_per_s", C.c_double)]


class mt_field_paths(C.Structure):
    _fields_ = [("records_per_launch", C.c_double), ("ldg_records_per_s", C.c_double),
                ("tex_records_per_s", C.c_double), ("tma_records_per_s", C.c_double)]


class mt_muons_in(C.Structure):
    _fields_ = [("pos_q", C.c_void_p), ("mom", C.c_void_p)]


class mt_muons_out(C.Structure):
    _fields_ = [("pos_flag", C.c_void_p), ("mom_steps", C.c_void_p), ("exit_rec", C.c_void_p),
                ("exit_count", C.c_void_p), ("exit_capacity", C.c_uint32), ("counters", C.c_void_p)]


_lib = None


def lib():
    """Load the C-ABI library; raise if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libmuon_transport.so is missing: run `python -m paper_2512_10520_b200.build` "
                               "(nvcc, sm_100a).  There is no CPU fallback.")
        L = C.CDLL(LIB_PATH)
        L.mt_strerror.restype = C.c_char_p
        L.mt_strerror.argtypes = [C.c_int]
        L.mt_last_error.restype = C.c_char_p
        L.mt_last_error.argtypes = [C.c_void_p]
        L.mt_create.argtypes = [C.POINTER(C.c_void_p), C.c_int]
        L.mt_destroy.argtypes = [C.c_void_p]
        L.mt_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int64]
        L.mt_load_histograms.argtypes = [C.c_void_p, C.POINTER(mt_hist_desc)]
        L.mt_build_alias.argtypes = [C.c_void_p, C.c_int]
        L.mt_get_alias.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.mt_set_geometry.argtypes = [C.c_void_p, C.POINTER(mt_geometry)]
        for name in ("mt_transport", "mt_transport_host", "mt_transport_static_scratch"):
            getattr(L, name).argtypes = [C.c_void_p, C.POINTER(mt_muons_in), C.c_uint64, C.c_uint64, C.c_uint64,
                                         C.POINTER(mt_muons_out), C.c_void_p]
        L.mt_launch_count.restype = C.c_int64
        L.mt_launch_count.argtypes = [C.c_void_p]
        L.mt_get_info.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int64)]
        L.mt_debug_sample.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_uint64, C.c_void_p, C.c_void_p]
        L.mt_debug_philox.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint64, C.c_void_p, C.c_void_p]
        L.mt_debug_lookup.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


_probes = None


def probes_lib():
    """Load libmuon_probes.so (include/muon_probes.h): measurement harness for bench.py and the tests, not the product."""
    global _probes
    if _probes is None:
        if not os.path.exists(PROBES_LIB_PATH):
            raise RuntimeError("libmuon_probes.so is missing: run `python -m paper_2512_10520_b200.build`")
        L = C.CDLL(PROBES_LIB_PATH)
        L.mt_measure_peaks.argtypes = [C.c_int, C.POINTER(mt_peaks)]
        L.mt_probe_field_paths.argtypes = [C.c_int, C.POINTER(mt_field_paths)]
        _probes = L
    return _probes


class MtError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("%s (%d): %s" % (lib().mt_strerror(code).decode(), code, text))
        self.code = code


def _check(ctx, rc):
    if rc != MT_OK:
        raise MtError(rc, lib().mt_last_error(ctx).decode() if ctx else "")


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _stream_ptr(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(getattr(stream, "cuda_stream", stream))


def _torch_stream(stream):
    """the torch view of `stream` (None = current stream, a torch stream, or a raw cudaStream_t value)"""
    import torch
    if stream is None:
        return torch.cuda.current_stream()
    if isinstance(stream, torch.cuda.Stream):
        return stream
    return torch.cuda.ExternalStream(int(stream))


# ------------------------------------------------------------------------------- the C calls, one to one
def mt_create(device=0):
    ctx = C.c_void_p()
    rc = lib().mt_create(C.byref(ctx), int(device))
    if rc != MT_OK:
        raise MtError(rc, "mt_create(device=%d): no usable CUDA device" % device)
    return ctx


def mt_destroy(ctx):
    _check(None, lib().mt_destroy(ctx))


def mt_set_option(ctx, option, value):
    _check(ctx, lib().mt_set_option(ctx, int(option), int(value)))


def mt_load_histograms(ctx, hist):
    """hist: workloads.Histograms (or any object with the same attributes); host arrays."""
    joint = bool(getattr(hist, "joint", False))
    keep = [_np(hist.counts_dp, np.float32), None if joint else _np(hist.counts_th, np.float32),
            _np(hist.axis_dp, np.float32), _np(hist.axis_th, np.float32), _np(hist.step_m, np.float32)]
    assert keep[0].size == hist.n_materials * hist.n_pbins * hist.n_dp * (hist.n_th if joint else 1)
    assert joint or keep[1].size == hist.n_materials * hist.n_pbins * hist.n_th
    assert keep[2].size == keep[3].size == hist.n_materials * hist.n_pbins * 2 and keep[4].size == hist.n_materials + 1
    d = mt_hist_desc(hist.n_materials, hist.n_pbins, hist.p_lo, hist.p_hi, hist.n_dp, hist.n_th,
                     *[a.ctypes.data if a is not None else None for a in keep],
                     MT_HIST_JOINT if joint else MT_HIST_MARGINAL)
    _check(ctx, lib().mt_load_histograms(ctx, C.byref(d)))


def mt_build_alias(ctx, placement=MT_PLACE_AUTO):
    _check(ctx, lib().mt_build_alias(ctx, int(placement)))


def mt_get_alias(ctx, hist):
    if getattr(hist, "joint", False):
        shp = (hist.n_materials, hist.n_pbins, hist.n_dp * hist.n_th)
        prob, alias = np.empty(shp, np.float32), np.empty(shp, np.uint32)
        _check(ctx, lib().mt_get_alias(ctx, prob.ctypes.data, alias.ctypes.data, None, None))
        return prob, alias, None, None
    shp_dp = (hist.n_materials, hist.n_pbins, hist.n_dp)
    shp_th = (hist.n_materials, hist.n_pbins, hist.n_th)
    prob_dp, alias_dp = np.empty(shp_dp, np.float32), np.empty(shp_dp, np.uint32)
    prob_th, alias_th = np.empty(shp_th, np.float32), np.empty(shp_th, np.uint32)
    _check(ctx, lib().mt_get_alias(ctx, prob_dp.ctypes.data, alias_dp.ctypes.data, prob_th.ctypes.data,
                                   alias_th.ctypes.data))
    return prob_dp, alias_dp, prob_th, alias_th


def mt_set_geometry(ctx, geom):
    """geom: workloads.Geometry; in voxel mode geom.material / geom.field are CUDA torch tensors."""
    g = mt_geometry()
    g.mode = geom.mode
    g.x_min, g.x_max, g.y_min, g.y_max, g.z_min, g.z_exit = geom.x_min, geom.x_max, geom.y_min, geom.y_max, geom.z_min, geom.z_exit
    g.p_min, g.max_steps, g.world_material = geom.p_min, geom.max_steps, geom.world_material
    g.field_mode = int(getattr(geom, "field_mode", 0))
    g.exit_mode = int(getattr(geom, "exit_mode", 0))
    keep = None
    if geom.mode == MT_GEOM_REGIONS:
        regs = np.ascontiguousarray(geom.regions) if geom.regions is not None else np.zeros(0, np.uint8)
        assert regs.size == 0 or regs.dtype.itemsize == C.sizeof(mt_region)
        keep = regs
        g.n_regions = len(regs)
        g.regions = regs.ctypes.data if len(regs) else None
    elif geom.mode == MT_GEOM_POLY:
        blocks = np.ascontiguousarray(geom.blocks) if geom.blocks is not None else np.zeros(0, np.uint8)
        assert blocks.size == 0 or blocks.dtype.itemsize == C.sizeof(mt_poly_block)
        keep = blocks
        g.n_blocks = len(blocks)
        g.blocks = blocks.ctypes.data if len(blocks) else None
    else:
        import torch
        mat, fld = geom.material, geom.field
        if not (isinstance(mat, torch.Tensor) and mat.is_cuda and isinstance(fld, torch.Tensor) and fld.is_cuda):
            raise ValueError("voxel grids must be CUDA torch tensors")
        mat, fld = mat.contiguous(), fld.contiguous()
        assert mat.dtype == torch.uint8 and fld.dtype == torch.float32
        assert tuple(mat.shape) == (geom.nz, geom.ny, geom.nx) and tuple(fld.shape) == (geom.nz, geom.ny, geom.nx, 3)
        keep = (mat, fld)
        g.nx, g.ny, g.nz = geom.nx, geom.ny, geom.nz
        g.ox, g.oy, g.oz, g.cell = geom.ox, geom.oy, geom.oz, geom.cell
        g.d_material, g.d_field = mat.data_ptr(), fld.data_ptr()
        torch.cuda.current_stream().synchronize()      # the library repacks on the default stream
    _check(ctx, lib().mt_set_geometry(ctx, C.byref(g)))
    del keep


def mt_transport(ctx, pos_q, mom, seed, id_base=0, out=None, exit_capacity=0, counters=True, stream=None,
                 count_exits=False):
    """pos_q, mom: CUDA float32 tensors [n,4].  Returns dict of CUDA tensors (asynchronous on the stream):
    pos_flag [n,4], mom_steps [n,4], and optionally exit_rec [cap,8], exit_count [1], counters [8].
    count_exits=True passes exit_count without a list (exit-plane hits are counted, no records written)."""
    import torch
    assert pos_q.is_cuda and mom.is_cuda and pos_q.dtype == torch.float32 and mom.dtype == torch.float32
    pos_q, mom = pos_q.contiguous(), mom.contiguous()
    n = pos_q.shape[0]
    assert tuple(pos_q.shape) == (n, 4) and tuple(mom.shape) == (n, 4)
    dev = pos_q.device
    if out is None:
        out = {}
    # the zero-fills below must be ordered before the kernels: they are enqueued on the stream the kernels run on
    with torch.cuda.stream(_torch_stream(stream)):
        if "pos_flag" not in out:
            out["pos_flag"] = torch.empty((n, 4), dtype=torch.float32, device=dev)
            out["mom_steps"] = torch.empty((n, 4), dtype=torch.float32, device=dev)
        if exit_capacity and "exit_rec" not in out:
            out["exit_rec"] = torch.zeros((exit_capacity, 8), dtype=torch.float32, device=dev)
        if "exit_rec" in out or count_exits:
            out["exit_count"] = torch.zeros(1, dtype=torch.int32, device=dev)
        if counters:
            out["counters"] = torch.zeros(8, dtype=torch.int64, device=dev)
    o = mt_muons_out()
    o.pos_flag, o.mom_steps = out["pos_flag"].data_ptr(), out["mom_steps"].data_ptr()
    if "exit_rec" in out:
        o.exit_rec, o.exit_count, o.exit_capacity = out["exit_rec"].data_ptr(), out["exit_count"].data_ptr(), out["exit_rec"].shape[0]
    elif count_exits:
        o.exit_count = out["exit_count"].data_ptr()
    if counters:
        o.counters = out["counters"].data_ptr()
    i = mt_muons_in(pos_q.data_ptr(), mom.data_ptr())
    _check(ctx, lib().mt_transport(ctx, C.byref(i), n, int(id_base), int(seed), C.byref(o), _stream_ptr(stream)))
    return out


def mt_transport_static_scratch(ctx, pos_q, mom, seed, out, id_base=0, stream=None):
    """mt_transport for a caller that must not allocate device memory (include/muon_transport.h has the full story):
    the library keeps the scratch of this call in a fixed array inside its own image, so at most
    MT_STATIC_SCRATCH_MAX_MUONS muons per call, and calls must not overlap on the GPU.  For the same reason nothing is
    allocated HERE either: `out` must already hold the caller's CUDA tensors "pos_flag" and "mom_steps" [n,4] float32 and
    may hold "exit_rec" [cap,8] float32 with "exit_count" [1] int32, "exit_count" alone, and "counters" [8] int64; the
    caller zeroes exit_count and counters (they are added to).  pos_q / mom must be contiguous.  Returns `out`."""
    import torch
    n = pos_q.shape[0]
    for t, shape in ((pos_q, (n, 4)), (mom, (n, 4)), (out["pos_flag"], (n, 4)), (out["mom_steps"], (n, 4))):
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == shape
    o = mt_muons_out()
    o.pos_flag, o.mom_steps = out["pos_flag"].data_ptr(), out["mom_steps"].data_ptr()
    if "exit_count" in out:
        o.exit_count = out["exit_count"].data_ptr()
    if "exit_rec" in out:
        o.exit_rec, o.exit_capacity = out["exit_rec"].data_ptr(), out["exit_rec"].shape[0]
    if "counters" in out:
        o.counters = out["counters"].data_ptr()
    i = mt_muons_in(pos_q.data_ptr(), mom.data_ptr())
    _check(ctx, lib().mt_transport_static_scratch(ctx, C.byref(i), n, int(id_base), int(seed), C.byref(o),
                                                  _stream_ptr(stream)))
    return out


def mt_transport_host(ctx, pos_q, mom, seed, id_base=0, out=None, exit_capacity=0, counters=True, stream=None):
    """Same call with HOST buffers (numpy arrays or pinned CPU torch tensors); returns numpy arrays."""
    pos_q, mom = _as_host(pos_q), _as_host(mom)
    n = pos_q.shape[0]
    if out is None:
        out = {"pos_flag": np.empty((n, 4), np.float32), "mom_steps": np.empty((n, 4), np.float32)}
    o = mt_muons_out()
    o.pos_flag, o.mom_steps = _host_ptr(out["pos_flag"]), _host_ptr(out["mom_steps"])
    if exit_capacity:
        out["exit_rec"] = np.zeros((exit_capacity, 8), np.float32)
        out["exit_count"] = np.zeros(1, np.uint32)
        o.exit_rec, o.exit_count, o.exit_capacity = out["exit_rec"].ctypes.data, out["exit_count"].ctypes.data, exit_capacity
    if counters:
        out["counters"] = np.zeros(8, np.uint64)
        o.counters = out["counters"].ctypes.data
    i = mt_muons_in(_host_ptr(pos_q), _host_ptr(mom))
    _check(ctx, lib().mt_transport_host(ctx, C.byref(i), n, int(id_base), int(seed), C.byref(o), _stream_ptr(stream)))
    return out


def _as_host(a):
    if hasattr(a, "data_ptr"):
        assert not a.is_cuda and a.is_contiguous()
        return a
    return _np(a, np.float32)


def _host_ptr(a):
    return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data


def mt_launch_count(ctx):
    return int(lib().mt_launch_count(ctx))


def mt_get_info(ctx, what):
    v = C.c_int64(0)
    rc = lib().mt_get_info(ctx, what, C.byref(v))
    if rc != MT_OK:
        raise MtError(rc, "mt_get_info")
    return int(v.value)


def mt_measure_peaks(device=0):
    """dict of the measured issue and gather peaks of the device (include/muon_probes.h: mt_peaks)"""
    p = mt_peaks()
    rc = probes_lib().mt_measure_peaks(int(device), C.byref(p))
    if rc != MT_OK:
        raise MtError(rc, "mt_measure_peaks(device=%d)" % device)
    return {name: getattr(p, name) for name, _ in mt_peaks._fields_}


def mt_probe_field_paths(device=0):
    """corner records per second through global loads / texture fetches / a TMA-staged shared-memory window"""
    p = mt_field_paths()
    rc = probes_lib().mt_probe_field_paths(int(device), C.byref(p))
    if rc != MT_OK:
        raise MtError(rc, "mt_probe_field_paths(device=%d)" % device)
    return {name: getattr(p, name) for name, _ in mt_field_paths._fields_}


def mt_debug_sample(ctx, material, pbin, which, words, stream=None, joint=False):
    """words: int32 CUDA tensor [n]; joint mode: [2n] = n select words then n accept words -> [n] cells"""
    import torch
    words = words.contiguous()
    assert words.is_cuda and words.dtype == torch.int32
    n = words.numel() // 2 if joint else words.numel()
    out = torch.empty(n, dtype=torch.int32, device=words.device)
    _check(ctx, lib().mt_debug_sample(ctx, material, pbin, which, words.data_ptr(), n, out.data_ptr(),
                                      _stream_ptr(stream)))
    return out


def mt_debug_lookup(ctx, xyz, stream=None):
    """xyz: float32 CUDA tensor [n,3] -> (material int32 [n], field float32 [n,3]) as the step loop looks them up"""
    import torch
    xyz = xyz.contiguous()
    assert xyz.is_cuda and xyz.dtype == torch.float32 and xyz.shape[-1] == 3
    n = xyz.shape[0]
    mat = torch.empty(n, dtype=torch.int32, device=xyz.device)
    fld = torch.empty((n, 3), dtype=torch.float32, device=xyz.device)
    _check(ctx, lib().mt_debug_lookup(ctx, xyz.data_ptr(), n, mat.data_ptr(), fld.data_ptr(), _stream_ptr(stream)))
    return mat, fld


def mt_debug_philox(ctx, seed, id_base, step, n, device="cuda", stream=None):
    import torch
    out = torch.empty((n, 4), dtype=torch.int32, device=device)
    _check(ctx, lib().mt_debug_philox(ctx, int(seed), int(id_base), int(step), n, out.data_ptr(), _stream_ptr(stream)))
    return out


class MuonTransport:
    """The four calls chained for one workload (workloads.Workload); owns the context."""

    def __init__(self, device=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the transport path has no CPU fallback")
        self.device = device
        self.ctx = mt_create(device)

    def setup(self, hist, geom, placement=MT_PLACE_AUTO):
        mt_load_histograms(self.ctx, hist)
        mt_build_alias(self.ctx, placement)
        mt_set_geometry(self.ctx, geom)
        return self

    def set_option(self, option, value):
        mt_set_option(self.ctx, option, value)
        return self

    def transport(self, pos_q, mom, seed, **kw):
        return mt_transport(self.ctx, pos_q, mom, seed, **kw)

    def transport_host(self, pos_q, mom, seed, **kw):
        return mt_transport_host(self.ctx, pos_q, mom, seed, **kw)

    def transport_static_scratch(self, pos_q, mom, seed, out, **kw):
        return mt_transport_static_scratch(self.ctx, pos_q, mom, seed, out, **kw)

    def close(self):
        if self.ctx is not None:
            mt_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
