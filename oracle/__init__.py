"""ctypes front end of the CPU oracle (TEST INFRASTRUCTURE ONLY).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports paper_2512_10520_b200 (the CUDA path), and the CUDA path never imports
it.  All arithmetic lives in muon_oracle.cpp; this file only marshals numpy arrays.
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

FLAG_STOPPED, FLAG_EXITED, FLAG_ESCAPED, FLAG_MAXSTEPS = 1, 2, 3, 4

_lib = None

REGION_DTYPE = np.dtype([("z_lo", "<f4"), ("z_hi", "<f4"), ("x_lo", "<f4"), ("x_hi", "<f4"),
                         ("y_lo", "<f4"), ("y_hi", "<f4"), ("material", "<i4"),
                         ("bx", "<f4"), ("by", "<f4"), ("bz", "<f4")])

# vertex i of the lower face is joined to vertex i of the upper face
POLY_DTYPE = np.dtype([("z_lo", "<f4"), ("z_hi", "<f4"), ("xy_lo", "<f4", (4, 2)), ("xy_hi", "<f4", (4, 2)),
                       ("material", "<i4"), ("bx", "<f4"), ("by", "<f4"), ("bz", "<f4")])


class _Geometry(C.Structure):
    _fields_ = [("mode", C.c_int32),
                ("x_min", C.c_float), ("x_max", C.c_float), ("y_min", C.c_float), ("y_max", C.c_float),
                ("z_min", C.c_float), ("z_exit", C.c_float),
                ("p_min", C.c_float), ("max_steps", C.c_int32), ("world_material", C.c_int32),
                ("n_regions", C.c_int32), ("regions", C.c_void_p),
                ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("ox", C.c_float), ("oy", C.c_float), ("oz", C.c_float), ("cell", C.c_float),
                ("material", C.c_void_p), ("field", C.c_void_p), ("field_mode", C.c_int32),
                ("n_blocks", C.c_int32), ("blocks", C.c_void_p)]


class _Tables(C.Structure):
    _fields_ = [("n_materials", C.c_int32), ("n_pbins", C.c_int32), ("n_dp", C.c_int32), ("n_th", C.c_int32),
                ("p_lo", C.c_double), ("p_hi", C.c_double),
                ("prob_dp", C.c_void_p), ("alias_dp", C.c_void_p),
                ("prob_th", C.c_void_p), ("alias_th", C.c_void_p),
                ("axis_dp", C.c_void_p), ("axis_th", C.c_void_p), ("step_m", C.c_void_p), ("joint", C.c_int32)]


def lib():
    global _lib
    if _lib is None:
        # MUON_ORACLE_LIB: an alternative build of the same source (oracle/build.py --sanitize) for the sanitizer run
        _lib = C.CDLL(os.environ.get("MUON_ORACLE_LIB") or _build())
        _lib.orc_kick_f64.restype = C.c_double
        _lib.orc_kick_f32.restype = C.c_float
        _lib.orc_kick_f64.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_uint32]
        _lib.orc_kick_f32.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_uint32]
        _lib.orc_kick_joint_f64.restype = C.c_double
        _lib.orc_kick_joint_f32.restype = C.c_float
        _lib.orc_kick_joint_f64.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_uint32]
        _lib.orc_kick_joint_f32.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_uint32]
        _lib.orc_rk4_f64.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_double, C.c_int]
        _lib.orc_rk4_f32.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_float, C.c_int]
        _lib.orc_make_edges.argtypes = [C.c_double, C.c_double, C.c_int, C.c_void_p]
        _lib.orc_muon_words.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_void_p]
        for name in ("orc_transport_f32", "orc_transport_f64", "orc_transport_libm_f32", "orc_transport_libm_f64"):
            getattr(_lib, name).argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint64, C.c_void_p,
                                            C.c_uint64] + [C.c_void_p] * 6 + [C.c_int]
        _lib.orc_trace_f32.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint64] + [C.c_void_p] * 7 + [C.c_int32]
    return _lib


def _p(a):
    return C.c_void_p(a.ctypes.data)


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def max_threads() -> int:
    return int(lib().orc_max_threads())


# ---------------------------------------------------------------------------------------------- RNG
def philox4x32_10(ctr, key):
    """ctr [n,4] uint32, key [2] uint32 -> [n,4] uint32"""
    ctr = _c(ctr, np.uint32).reshape(-1, 4)
    key = _c(key, np.uint32)
    out = np.empty_like(ctr)
    lib().orc_philox4x32_10(_p(ctr), _p(key), _p(out), C.c_uint64(len(ctr)))
    return out


def muon_words(seed, muon_id, step):
    w = np.empty(4, np.uint32)
    lib().orc_muon_words(seed, muon_id, step, _p(w))
    return w


# ------------------------------------------------------------------------------------------- tables
def build_alias(counts):
    """counts [..., N] float32 -> (prob float32, alias uint32) of the same shape"""
    counts = _c(counts, np.float32)
    N = counts.shape[-1]
    flat = counts.reshape(-1, N)
    prob = np.empty_like(flat)
    alias = np.empty(flat.shape, np.uint32)
    rc = lib().orc_build_alias(_p(flat), C.c_int(flat.shape[0]), C.c_int(N), _p(prob), _p(alias))
    if rc != 0:
        raise ValueError("empty or invalid histogram at table %d" % (-rc - 1))
    return prob.reshape(counts.shape), alias.reshape(counts.shape)


def alias_draw(prob, alias, words):
    prob, alias, words = _c(prob, np.float32), _c(alias, np.uint32), _c(words, np.uint32)
    out = np.empty(words.shape, np.uint32)
    lib().orc_alias_draw(_p(prob), _p(alias), C.c_int(len(prob)), _p(words), C.c_uint64(words.size), _p(out))
    return out


def alias_draw2(prob, alias, w_sel, w_acc):
    """two-word draw of the joint mode"""
    prob, alias = _c(prob, np.float32).reshape(-1), _c(alias, np.uint32).reshape(-1)
    w_sel, w_acc = _c(w_sel, np.uint32), _c(w_acc, np.uint32)
    out = np.empty(w_sel.shape, np.uint32)
    lib().orc_alias_draw2(_p(prob), _p(alias), C.c_uint32(len(prob)), _p(w_sel), _p(w_acc), C.c_uint64(w_sel.size), _p(out))
    return out


def alias_enumerate(prob, alias):
    """exact outcome counts over all 2^32 words (use only for tiny N; ~10 s)"""
    prob, alias = _c(prob, np.float32), _c(alias, np.uint32)
    out = np.zeros(len(prob), np.uint64)
    lib().orc_alias_enumerate(_p(prob), _p(alias), C.c_int(len(prob)), _p(out))
    return out


def make_edges(p_lo, p_hi, n):
    e = np.empty(n + 1, np.float32)
    lib().orc_make_edges(p_lo, p_hi, n, _p(e))
    return e


def momentum_bin(edges, P):
    edges, P = _c(edges, np.float32), _c(P, np.float32)
    out = np.empty(P.shape, np.int32)
    lib().orc_momentum_bin(_p(edges), C.c_int(len(edges) - 1), _p(P), C.c_uint64(P.size), _p(out))
    return out


# ---------------------------------------------------------------------------------- transcendentals
def exp2c(y):
    y = _c(y, np.float32)
    out = np.empty_like(y)
    lib().orc_exp2c_f32(_p(y), C.c_uint64(y.size), _p(out))
    return out


def sincos_polar(theta):
    theta = _c(theta, np.float32)
    s, c = np.empty_like(theta), np.empty_like(theta)
    lib().orc_sincos_polar_f32(_p(theta), C.c_uint64(theta.size), _p(s), _p(c))
    return s, c


def sincos_azimuth(k24):
    k24 = _c(k24, np.uint32)
    s, c = np.empty(k24.shape, np.float32), np.empty(k24.shape, np.float32)
    lib().orc_sincos_azimuth_f32(_p(k24), C.c_uint64(k24.size), _p(s), _p(c))
    return s, c


# ------------------------------------------------------------------------------------ kick, RK4
def frame(d, dtype=np.float64):
    d = _c(d, dtype)
    e1, e2 = np.empty(3, dtype), np.empty(3, dtype)
    (lib().orc_frame_f64 if dtype == np.float64 else lib().orc_frame_f32)(_p(d), _p(e1), _p(e2))
    return e1, e2


def kick(p, f, theta, k24, dtype=np.float64):
    """one sampling kick -> (new p, Pn)"""
    p = _c(p, dtype).copy()
    P = np.sqrt((p.astype(np.float64) ** 2).sum())
    if dtype == np.float64:
        Pn = lib().orc_kick_f64(_p(p), float(P), float(f), float(theta), int(k24))
    else:
        Pn = lib().orc_kick_f32(_p(p), float(np.float32(P)), float(np.float32(f)), float(np.float32(theta)), int(k24))
    return p, Pn


def kick_joint(p, fz, ft, k24, dtype=np.float64):
    """one kick of the joint mode -> (new p, new |p|)"""
    p = _c(p, dtype).copy()
    P = np.sqrt((p.astype(np.float64) ** 2).sum())
    if dtype == np.float64:
        Pn = lib().orc_kick_joint_f64(_p(p), float(P), float(fz), float(ft), int(k24))
    else:
        Pn = lib().orc_kick_joint_f32(_p(p), float(np.float32(P)), float(np.float32(fz)), float(np.float32(ft)), int(k24))
    return p, Pn


def rk4(r, p, q, B, h, n_steps, dtype=np.float64):
    """n_steps RK4 steps of length h in a uniform field B -> (r, p)"""
    r, p, B = _c(r, dtype).copy(), _c(p, dtype).copy(), _c(B, dtype)
    if dtype == np.float64:
        lib().orc_rk4_f64(_p(r), _p(p), float(q), _p(B), float(h), int(n_steps))
    else:
        lib().orc_rk4_f32(_p(r), _p(p), float(q), _p(B), float(h), int(n_steps))
    return r, p


# ----------------------------------------------------------------------------------------- geometry
def _host(a, dtype):
    if a is None:
        return None
    if hasattr(a, "detach"):      # torch tensor (possibly on a GPU)
        a = a.detach().cpu().numpy()
    return np.ascontiguousarray(a, dtype=dtype)


class OracleGeometry:
    """Host copy of a workloads.Geometry in the oracle's own struct layout."""

    def __init__(self, g):
        self.regions = _c(g.regions, REGION_DTYPE) if g.regions is not None else np.zeros(0, REGION_DTYPE)
        self.material = _host(g.material, np.uint8)
        self.field = _host(g.field, np.float32)
        s = _Geometry()
        s.mode = g.mode
        s.x_min, s.x_max, s.y_min, s.y_max, s.z_min, s.z_exit = g.x_min, g.x_max, g.y_min, g.y_max, g.z_min, g.z_exit
        s.p_min, s.max_steps, s.world_material = g.p_min, g.max_steps, g.world_material
        s.n_regions = len(self.regions)
        s.regions = self.regions.ctypes.data if len(self.regions) else None
        s.nx, s.ny, s.nz = g.nx, g.ny, g.nz
        s.ox, s.oy, s.oz, s.cell = g.ox, g.oy, g.oz, g.cell
        s.material = self.material.ctypes.data if self.material is not None else None
        s.field = self.field.ctypes.data if self.field is not None else None
        s.field_mode = int(getattr(g, "field_mode", 0))
        blocks = getattr(g, "blocks", None)
        self.blocks = _c(blocks, POLY_DTYPE) if blocks is not None else np.zeros(0, POLY_DTYPE)
        s.n_blocks = len(self.blocks)
        s.blocks = self.blocks.ctypes.data if len(self.blocks) else None
        self.struct = s


def material_and_field(geom, xyz, dtype=np.float32):
    og = geom if isinstance(geom, OracleGeometry) else OracleGeometry(geom)
    xyz = _c(xyz, dtype).reshape(-1, 3)
    mat = np.empty(len(xyz), np.int32)
    B = np.empty((len(xyz), 3), dtype)
    fn = lib().orc_material_and_field_f64 if dtype == np.float64 else lib().orc_material_and_field_f32
    fn(C.byref(og.struct), _p(xyz), C.c_uint64(len(xyz)), _p(mat), _p(B))
    return mat, B


class OracleTables:
    """Alias tables built by the oracle's own construction from a workloads.Histograms."""

    def __init__(self, h):
        self.h = h
        self.joint = bool(getattr(h, "joint", False))
        if self.joint:       # counts_dp holds the joint histograms [M][nb][n_dp][n_th]; one table per (M, i)
            flat = _c(h.counts_dp, np.float32).reshape(h.n_materials, h.n_pbins, h.n_dp * h.n_th)
            self.prob_dp, self.alias_dp = build_alias(flat)
            self.prob_th, self.alias_th = np.zeros(1, np.float32), np.zeros(1, np.uint32)
        else:
            self.prob_dp, self.alias_dp = build_alias(h.counts_dp)
            self.prob_th, self.alias_th = build_alias(h.counts_th)
        self.axis_dp, self.axis_th = _c(h.axis_dp, np.float32), _c(h.axis_th, np.float32)
        self.step_m = _c(h.step_m, np.float32)
        s = _Tables()
        s.n_materials, s.n_pbins, s.n_dp, s.n_th = h.n_materials, h.n_pbins, h.n_dp, h.n_th
        s.p_lo, s.p_hi = float(np.float32(h.p_lo)), float(np.float32(h.p_hi))
        s.prob_dp, s.alias_dp = self.prob_dp.ctypes.data, self.alias_dp.ctypes.data
        s.prob_th, s.alias_th = self.prob_th.ctypes.data, self.alias_th.ctypes.data
        s.axis_dp, s.axis_th, s.step_m = self.axis_dp.ctypes.data, self.axis_th.ctypes.data, self.step_m.ctypes.data
        s.joint = 1 if self.joint else 0
        self.struct = s

    @property
    def edges(self):
        return make_edges(self.struct.p_lo, self.struct.p_hi, self.h.n_pbins)


def transport(tables, geom, pos_q, mom, seed, id_base=0, ids=None, dtype=np.float32, threads=1, libm=False):
    """Algorithm 1 for every muon.  pos_q [n,4] = x,y,z,q; mom [n,4] = px,py,pz,-.

    libm=True: the witness mode — the C library's exp2 / sin / cos in place of the fixed polynomials of DESIGN.md
    §3.6 (not the parity reference: used to exercise north_star's tolerance against the plain definitions).
    Returns dict(pos [n,3], mom [n,3], flag [n] int32, steps [n] int32) in `dtype`."""
    og = geom if isinstance(geom, OracleGeometry) else OracleGeometry(geom)
    pos_q, mom = _c(pos_q, dtype).reshape(-1, 4), _c(mom, dtype).reshape(-1, 4)
    n = len(pos_q)
    out_pos, out_mom = np.empty((n, 3), dtype), np.empty((n, 3), dtype)
    flag, steps = np.empty(n, np.int32), np.empty(n, np.int32)
    ids_arr = _c(ids, np.uint64) if ids is not None else None
    fn = getattr(lib(), "orc_transport_%s%s" % ("libm_" if libm else "", "f64" if dtype == np.float64 else "f32"))
    rc = fn(C.byref(tables.struct), C.byref(og.struct), seed, id_base,
            _p(ids_arr) if ids_arr is not None else None, n,
            _p(pos_q), _p(mom), _p(out_pos), _p(out_mom), _p(flag), _p(steps), int(threads))
    assert rc == 0
    return dict(pos=out_pos, mom=out_mom, flag=flag, steps=steps)


def exit_project(pos, mom, z_exit, dtype=np.float32):
    """positions [n,3] of EXITED muons projected back onto the plane z = z_exit along mom [n,3]."""
    pos = np.array(_c(pos, dtype).reshape(-1, 3), copy=True)
    mom = _c(mom, dtype).reshape(-1, 3)
    if dtype == np.float64:
        lib().orc_exit_project_f64(_p(pos), _p(mom), C.c_uint64(len(pos)), C.c_double(z_exit))
    else:
        lib().orc_exit_project_f32(_p(pos), _p(mom), C.c_uint64(len(pos)), C.c_float(z_exit))
    return pos


def trace(tables, geom, pos_q, mom, seed, muon_id, cap=20000):
    """one muon in float32 with its per-step (material, pbin, cell_dp, cell_th) record"""
    og = geom if isinstance(geom, OracleGeometry) else OracleGeometry(geom)
    pos_q, mom = _c(pos_q, np.float32).reshape(4), _c(mom, np.float32).reshape(4)
    out_pos, out_mom = np.empty(3, np.float32), np.empty(3, np.float32)
    flag, steps = np.zeros(1, np.int32), np.zeros(1, np.int32)
    tr = np.full((cap, 4), -1, np.int32)
    lib().orc_trace_f32(C.byref(tables.struct), C.byref(og.struct), seed, muon_id, _p(pos_q), _p(mom),
                        _p(out_pos), _p(out_mom), _p(flag), _p(steps), _p(tr), cap)
    n = min(int(steps[0]), cap)
    return dict(pos=out_pos, mom=out_mom, flag=int(flag[0]), steps=int(steps[0]), trace=tr[:n])
