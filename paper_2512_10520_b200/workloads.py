"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: no alias tables, no Philox transport streams, no stepping.  It only draws histograms, muon
spectra, region lists and voxel grids with numpy's own generators.  It imports neither the binding nor
oracle/.  The paper's Geant4 histograms, SHiP geometry and field map are not
available; these inputs take their shapes and stand in for them.
"""
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field as _field
import math
import os

import numpy as np

REGION_DTYPE = np.dtype([("z_lo", "<f4"), ("z_hi", "<f4"), ("x_lo", "<f4"), ("x_hi", "<f4"),
                         ("y_lo", "<f4"), ("y_hi", "<f4"), ("material", "<i4"),
                         ("bx", "<f4"), ("by", "<f4"), ("bz", "<f4")])

# convex-polyhedra block: two quadrilateral faces, vertex i joined to vertex i
POLY_DTYPE = np.dtype([("z_lo", "<f4"), ("z_hi", "<f4"), ("xy_lo", "<f4", (4, 2)), ("xy_hi", "<f4", (4, 2)),
                       ("material", "<i4"), ("bx", "<f4"), ("by", "<f4"), ("bz", "<f4")])

MODE_REGIONS, MODE_VOXEL, MODE_POLY = 0, 1, 2
FIELD_TRILINEAR, FIELD_NEAREST, FIELD_PER_STAGE = 0, 1, 2

# material -> (density g/cm3, radiation length cm); BASELINE.json configs[0], configs[2]
MATERIALS = {"iron": (7.874, 1.757), "concrete": (2.3, 11.55), "air": (1.205e-3, 30390.0)}

_GEN_KEY = 0x4D54  # "MT": generator streams are numpy Philox(key=[_GEN_KEY + config, tag])


@dataclass
class Histograms:
    n_materials: int
    n_pbins: int
    n_dp: int
    n_th: int
    p_lo: float
    p_hi: float
    counts_dp: np.ndarray   # [n_materials][n_pbins][n_dp] float32
    counts_th: np.ndarray   # [n_materials][n_pbins][n_th] float32
    axis_dp: np.ndarray     # [n_materials][n_pbins][2] float32 = {log2 lower edge, log2 width per cell}
    axis_th: np.ndarray
    step_m: np.ndarray      # [n_materials + 1] float32, path length per step; index 0 = vacuum
    joint: bool = False     # True: counts_dp is ONE joint histogram [n_materials][n_pbins][n_dp][n_th] per (M, i) over
                            # (log2 of -dPz/|P|, log2 of dPt/|P|) as in PAPER.md L77, and counts_th is None


@dataclass
class Geometry:
    mode: int
    x_min: float
    x_max: float
    y_min: float
    y_max: float
    z_min: float
    z_exit: float
    p_min: float
    max_steps: int
    world_material: int
    regions: np.ndarray = None          # REGION_DTYPE, sorted by z_lo, z-disjoint
    nx: int = 0
    ny: int = 0
    nz: int = 0
    ox: float = 0.0
    oy: float = 0.0
    oz: float = 0.0
    cell: float = 0.0
    material: object = None             # uint8 [nz][ny][nx], numpy or torch (any device)
    field: object = None                # float32 [nz][ny][nx][3]
    field_mode: int = 0                 # FIELD_NEAREST | FIELD_PER_STAGE; 0 = trilinear, frozen
    blocks: np.ndarray = None           # POLY_DTYPE (MODE_POLY); the first block that contains a point wins
    exit_mode: int = 0                  # 1: the compact exit list is projected back onto the exit plane


@dataclass
class Muons:
    pos_q: np.ndarray                   # [n][4] float32: x, y, z (m), charge (+1/-1)
    mom: np.ndarray                     # [n][4] float32: px, py, pz (GeV/c), 0


@dataclass
class Workload:
    name: str
    hist: Histograms
    geom: Geometry
    muons: Muons
    seed: int = 1
    notes: dict = _field(default_factory=dict)


def _rng(config, tag):
    return np.random.Generator(np.random.Philox(key=[_GEN_KEY + config, tag]))


# --------------------------------------------------------------------------------------- histograms
def _one_histogram(args):
    (config, tag, rho, x0_cm, step_cm, p_a, p_b, n_dp, n_th, n_draws, joint) = args
    rng = _rng(config, tag)
    P = rng.uniform(p_a, p_b, n_draws)                                     # GeV
    # momentum loss: Moyal(loc, 0.1 loc) + Exp(mean 3e-6 rho L P)   [GeV]
    loc = 1.5e-3 * rho * step_cm
    z = rng.standard_normal(n_draws)
    moyal = -np.log(np.maximum(z * z, 1e-300))                             # Moyal(0,1) = -ln(Z^2)
    dp = loc + 0.1 * loc * moyal + rng.exponential(1.0, n_draws) * (3e-6 * rho * step_cm) * P
    f = dp / P
    # polar angle: |N(0, theta0)| with 1% from pdf ~ theta^-4 on [theta0, 10 theta0]
    lx = step_cm / x0_cm
    theta0 = 13.6e-3 / P * math.sqrt(lx) * (1.0 + 0.038 * math.log(lx))
    th = np.abs(theta0 * rng.standard_normal(n_draws))
    tail = rng.random(n_draws) < 0.01
    u = rng.random(n_draws)
    th = np.where(tail, theta0 * (1.0 - 0.999 * u) ** (-1.0 / 3.0), th)
    if joint:
        # the paper's variables (L73, L77): longitudinal fractional loss and transverse fractional kick of the
        # same draw, fz = -dPz/|P| = 1 - (1 - f) cos(theta), ft = dPt/|P| = (1 - f) sin(theta)
        f = np.minimum(f, 0.999)
        f, th = 1.0 - (1.0 - f) * np.cos(th), (1.0 - f) * np.sin(th)
    out, cells = [], []
    for v, n_cells, q_lo in ((f, n_dp, 0.0), (th, n_th, 1e-3)):
        lv = np.log2(np.maximum(v, 1e-300))
        lo = float(np.quantile(lv, q_lo)) if q_lo > 0 else float(lv.min())
        hi = float(np.nextafter(np.float32(lv.max()), np.float32(np.inf)))
        lo32 = np.float32(lo)
        d32 = np.float32((hi - float(lo32)) / n_cells)
        cell = np.clip(np.floor((lv - float(lo32)) / float(d32)), 0, n_cells - 1).astype(np.int64)
        counts = np.bincount(cell, minlength=n_cells).astype(np.float32)
        out.append((counts, np.array([lo32, d32], np.float32)))
        cells.append(cell)
    if joint:
        both = np.bincount(cells[0] * n_th + cells[1], minlength=n_dp * n_th).astype(np.float32)
        out[0] = (both.reshape(n_dp, n_th), out[0][1])
    return out


def make_histograms(config, materials, steps_cm, n_pbins, p_lo, p_hi, n_dp, n_th, n_draws=1_000_000,
                    vacuum_step_m=None, workers=None, joint=False):
    """materials: list of names (material id = index + 1); steps_cm: step length per material."""
    M = len(materials)
    edges = p_lo * (p_hi / p_lo) ** (np.arange(n_pbins + 1) / n_pbins)
    jobs = []
    for m, (name, step_cm) in enumerate(zip(materials, steps_cm)):
        rho, x0 = MATERIALS[name]
        for i in range(n_pbins):
            jobs.append((config, m * 4096 + i, rho, x0, step_cm, edges[i], edges[i + 1], n_dp, n_th, n_draws, joint))
    # MT_GEN_WORKERS: set by launchers that run several generating processes on one host (bench.py --gpus N)
    workers = workers or int(os.environ.get("MT_GEN_WORKERS", 0)) or min(32, os.cpu_count() or 1)
    with ThreadPoolExecutor(workers) as ex:
        res = list(ex.map(_one_histogram, jobs))
    counts_dp = np.stack([r[0][0] for r in res]).reshape((M, n_pbins, n_dp, n_th) if joint else (M, n_pbins, n_dp))
    counts_th = None if joint else np.stack([r[1][0] for r in res]).reshape(M, n_pbins, n_th)
    axis_dp = np.stack([r[0][1] for r in res]).reshape(M, n_pbins, 2)
    axis_th = np.stack([r[1][1] for r in res]).reshape(M, n_pbins, 2)
    step_m = np.array([vacuum_step_m if vacuum_step_m is not None else max(steps_cm) / 100.0]
                      + [s / 100.0 for s in steps_cm], np.float32)
    return Histograms(M, n_pbins, n_dp, n_th, float(p_lo), float(p_hi), counts_dp, counts_th,
                      axis_dp, axis_th, step_m, joint=joint)


# -------------------------------------------------------------------------------------------- muons
def spectrum_muons(config, n, xy="gauss", batch=0):
    """configs[1] spectrum: P ~ P^-2.7 on [10, 350] GeV, pT ~ Exp(0.5 GeV) (clipped to 0.9 P), uniform
    azimuth; charge +1 for even id, -1 for odd; x,y ~ N(0, 5 cm) ('gauss') or U(-0.5, 0.5) ('square')."""
    rng = _rng(config, 0x100000 + batch)
    u = rng.random(n)
    g = -1.7
    a, b = 10.0 ** g, 350.0 ** g
    P = (a + u * (b - a)) ** (1.0 / g)
    pt = np.minimum(rng.exponential(0.5, n), 0.9 * P)
    phi = rng.uniform(0.0, 2 * math.pi, n)
    pz = np.sqrt(P * P - pt * pt)
    if xy == "gauss":
        x, y = rng.normal(0.0, 0.05, n), rng.normal(0.0, 0.05, n)
    else:
        x, y = rng.uniform(-0.5, 0.5, n), rng.uniform(-0.5, 0.5, n)
    q = np.where(np.arange(n) % 2 == 0, 1.0, -1.0)
    pos_q = np.stack([x, y, np.zeros(n), q], 1).astype(np.float32)
    mom = np.stack([pt * np.cos(phi), pt * np.sin(phi), pz, np.zeros(n)], 1).astype(np.float32)
    return Muons(pos_q, mom)


# ----------------------------------------------------------------------------------------- geometry
def shield_regions(n_cells=8):
    """configs[2]: per 3.75 m cell: iron magnet 2.75 m (|x|,|y| < 0.6, By = +/-1.7 T alternating),
    air 0.25, concrete 0.5 (full xy), air 0.25.  Materials: 1 iron, 2 concrete, 3 air."""
    regs = []
    for c in range(n_cells):
        z0 = 3.75 * c
        by = 1.7 if c % 2 == 0 else -1.7
        regs.append((z0, z0 + 2.75, -0.6, 0.6, -0.6, 0.6, 1, 0.0, by, 0.0))
        regs.append((z0 + 2.75, z0 + 3.0, -1.0, 1.0, -1.0, 1.0, 3, 0.0, 0.0, 0.0))
        regs.append((z0 + 3.0, z0 + 3.5, -1.0, 1.0, -1.0, 1.0, 2, 0.0, 0.0, 0.0))
        regs.append((z0 + 3.5, z0 + 3.75, -1.0, 1.0, -1.0, 1.0, 3, 0.0, 0.0, 0.0))
    return np.array(regs, REGION_DTYPE)


def rasterise(regions, world_material, nx, ny, nz, ox, oy, oz, cell, config, device="cpu",
              n_modes=16, amplitude=0.1):
    """configs[3]: voxel material (cell-centre test against the boxes) and field = box field +
    (amplitude/n_modes) * sum_m a_m cos(2 pi k_m.r + phi_m).  Returns torch tensors on `device`."""
    import torch
    dev = torch.device(device)
    xc = torch.tensor(ox + (np.arange(nx) + 0.5) * cell, dtype=torch.float32, device=dev)
    yc = torch.tensor(oy + (np.arange(ny) + 0.5) * cell, dtype=torch.float32, device=dev)
    zc = torch.tensor(oz + (np.arange(nz) + 0.5) * cell, dtype=torch.float32, device=dev)
    material = torch.full((nz, ny, nx), world_material, dtype=torch.uint8, device=dev)
    fld = torch.zeros((nz, ny, nx, 3), dtype=torch.float32, device=dev)
    for r in regions:
        mz = (zc >= float(r["z_lo"])) & (zc < float(r["z_hi"]))
        my = (yc >= float(r["y_lo"])) & (yc < float(r["y_hi"]))
        mx = (xc >= float(r["x_lo"])) & (xc < float(r["x_hi"]))
        iz = torch.nonzero(mz).flatten()
        if iz.numel() == 0:
            continue
        z_a, z_b = int(iz[0]), int(iz[-1]) + 1
        m2 = (my[:, None] & mx[None, :])
        sub = material[z_a:z_b]
        sub[:, m2] = int(r["material"])
        fsub = fld[z_a:z_b]
        for c, key in enumerate(("bx", "by", "bz")):
            if float(r[key]) != 0.0:
                fsub[:, :, :, c][:, m2] = float(r[key])
    rng = _rng(config, 0x200000)
    a = rng.standard_normal((n_modes, 3))
    a /= np.linalg.norm(a, axis=1, keepdims=True)
    k = rng.uniform(-2.0, 2.0, (n_modes, 3))
    ph = rng.uniform(0.0, 2 * math.pi, n_modes)
    x64, y64, z64 = (ox + (np.arange(nx) + 0.5) * cell, oy + (np.arange(ny) + 0.5) * cell,
                     oz + (np.arange(nz) + 0.5) * cell)
    for m in range(n_modes):
        # cos(A + B), A = 2 pi (kx x + ky y) on the xy plane, B = 2 pi kz z + phi along z
        A = 2 * math.pi * (k[m, 0] * x64[None, :] + k[m, 1] * y64[:, None])
        Bz = 2 * math.pi * k[m, 2] * z64 + ph[m]
        cA = torch.tensor(np.cos(A), dtype=torch.float32, device=dev)
        sA = torch.tensor(np.sin(A), dtype=torch.float32, device=dev)
        cB = torch.tensor(np.cos(Bz), dtype=torch.float32, device=dev)
        sB = torch.tensor(np.sin(Bz), dtype=torch.float32, device=dev)
        wave = cB[:, None, None] * cA[None] - sB[:, None, None] * sA[None]
        for c in range(3):
            fld[..., c].add_(wave, alpha=float(amplitude / n_modes * a[m, c]))
        del wave
    return material, fld


# ---------------------------------------------------------------------------------------- configs
def config0(n=4096, n_draws=1_000_000, joint=False):
    """Toy slab, no field (BASELINE.json configs[0]).  joint=True: the paper's joint 2D histograms (§8(f) row 1)."""
    hist = make_histograms(0, ["iron"], [2.0], 50, 1.0, 300.0, 128, 64, n_draws, joint=joint)
    regs = np.array([(0.0, 1.0, -10.0, 10.0, -10.0, 10.0, 1, 0.0, 0.0, 0.0)], REGION_DTYPE)
    geom = Geometry(MODE_REGIONS, -10.0, 10.0, -10.0, 10.0, 0.0, 1.0, 1.0, 200, 0, regions=regs)
    pos_q = np.zeros((n, 4), np.float32)
    pos_q[:, 3] = -1.0
    mom = np.zeros((n, 4), np.float32)
    mom[:, 2] = 50.0
    return Workload("config0_toy_slab", hist, geom, Muons(pos_q, mom), seed=1)


def config1(n=65536, n_draws=1_000_000, joint=False):
    """Magnetised iron block (configs[1])."""
    hist = make_histograms(0, ["iron"], [2.0], 50, 1.0, 300.0, 128, 64, n_draws, joint=joint)
    regs = np.array([(0.0, 6.0, -1.0, 1.0, -1.0, 1.0, 1, 0.0, 1.7, 0.0)], REGION_DTYPE)
    geom = Geometry(MODE_REGIONS, -1.0, 1.0, -1.0, 1.0, 0.0, 6.0, 1.0, 1200, 0, regions=regs)
    return Workload("config1_magnetised_block", hist, geom, spectrum_muons(1, n, "gauss"), seed=1)


def shield_histograms(config, steps_cm, n_pbins=100, n_dp=256, n_th=128, n_draws=1_000_000, joint=False):
    return make_histograms(config, ["iron", "concrete", "air"], steps_cm, n_pbins, 1.0, 300.0, n_dp, n_th,
                           n_draws, joint=joint)


def config2(n=1_000_000, n_draws=1_000_000, n_cells=8, joint=False, table_shape=(100, 256, 128)):
    """Multi-region shield (configs[2]): sorted z-interval table plus per-region xy bounds."""
    hist = shield_histograms(2, [2.0, 2.0, 2.0], table_shape[0], table_shape[1], table_shape[2], n_draws, joint=joint)
    z_exit = 3.75 * n_cells
    geom = Geometry(MODE_REGIONS, -1.0, 1.0, -1.0, 1.0, 0.0, z_exit, 1.0, 6000, 3,
                    regions=shield_regions(n_cells))
    return Workload("config2_multi_region_shield", hist, geom, spectrum_muons(2, n, "square"), seed=1)


def regions_as_blocks(regions):
    """The same boxes written as polyhedra blocks (rectangular faces, counter-clockwise)."""
    out = np.zeros(len(regions), POLY_DTYPE)
    for b, r in zip(out, regions):
        rect = [(r["x_lo"], r["y_lo"]), (r["x_hi"], r["y_lo"]), (r["x_hi"], r["y_hi"]), (r["x_lo"], r["y_hi"])]
        b["z_lo"], b["z_hi"], b["xy_lo"], b["xy_hi"] = r["z_lo"], r["z_hi"], rect, rect
        b["material"], b["bx"], b["by"], b["bz"] = r["material"], r["bx"], r["by"], r["bz"]
    return out


def shield_polyhedra(n_cells=8):
    """A tapered-magnet shield in the shape of the paper's own geometry ("a sequence of
    magnets composed of iron blocks ... walls made of concrete"): per 3.75 m cell an iron core whose half-width in x
    tapers 0.25 -> 0.45 m (even cells) or 0.45 -> 0.25 m (odd cells) and whose half-height tapers 0.5 -> 0.6 m,
    By = +/-1.7 T alternating; two iron return yokes beside it (from 2 cm outside the core to twice its width) with the
    opposite field; a 0.5 m concrete wall (full xy).  Air is the world material.  The -x yokes are listed clockwise, the
    rest counter-clockwise.  Materials: 1 iron, 2 concrete, 3 air."""
    blocks = []

    def quad(x0, x1, y0, y1, clockwise=False):
        q = [(x0, y0), (x1, y0), (x1, y1), (x0, y1)]
        return q[::-1] if clockwise else q

    for c in range(n_cells):
        z0 = 3.75 * c
        by = 1.7 if c % 2 == 0 else -1.7
        w = (0.25, 0.45) if c % 2 == 0 else (0.45, 0.25)
        hh = (0.5, 0.6)
        gap = 0.02
        blocks.append((z0, z0 + 2.75, quad(-w[0], w[0], -hh[0], hh[0]), quad(-w[1], w[1], -hh[1], hh[1]), 1, 0.0, by, 0.0))
        blocks.append((z0, z0 + 2.75, quad(w[0] + gap, 2 * w[0] + gap, -hh[0], hh[0]),
                       quad(w[1] + gap, 2 * w[1] + gap, -hh[1], hh[1]), 1, 0.0, -by, 0.0))
        blocks.append((z0, z0 + 2.75, quad(-2 * w[0] - gap, -w[0] - gap, -hh[0], hh[0], True),
                       quad(-2 * w[1] - gap, -w[1] - gap, -hh[1], hh[1], True), 1, 0.0, -by, 0.0))
        blocks.append((z0 + 3.0, z0 + 3.5, quad(-1.0, 1.0, -1.0, 1.0), quad(-1.0, 1.0, -1.0, 1.0), 2, 0.0, 0.0, 0.0))
    return np.array(blocks, POLY_DTYPE)


def config2p(n=1_000_000, n_draws=1_000_000, n_cells=8, joint=False, table_shape=(100, 256, 128), field_mode=0):
    """Polyhedral shield: config 2's muons and histograms in the tapered-magnet geometry of
    shield_polyhedra(), looked up with the paper's slice + Eq. 2 test."""
    hist = shield_histograms(2, [2.0, 2.0, 2.0], table_shape[0], table_shape[1], table_shape[2], n_draws, joint=joint)
    geom = Geometry(MODE_POLY, -1.0, 1.0, -1.0, 1.0, 0.0, 3.75 * n_cells, 1.0, 6000, 3,
                    blocks=shield_polyhedra(n_cells), field_mode=field_mode)
    return Workload("config2p_polyhedral_shield", hist, geom, spectrum_muons(2, n, "square"), seed=1)


def config3(n=10_000_000, n_draws=1_000_000, n_cells=8, half_width_cells=100, device="cpu", hist=None,
            table_shape=(100, 256, 128), joint=False, field_mode=0):
    """Field-map shield (configs[3]): voxel material + trilinear field grid, 1 cm cells; steps 1 cm in
    iron and concrete, 10 cm in air.  `n_cells` / `half_width_cells` shrink the grid for CPU tests."""
    if hist is None:
        hist = shield_histograms(3, [1.0, 1.0, 10.0], table_shape[0], table_shape[1], table_shape[2], n_draws,
                                 joint=joint)
    cell = 0.01
    nx = ny = 2 * half_width_cells
    nz = int(round(3.75 * n_cells / cell))
    half = half_width_cells * cell
    material, fld = rasterise(shield_regions(n_cells), 3, nx, ny, nz, -half, -half, 0.0, cell, 3, device)
    geom = Geometry(MODE_VOXEL, -half, half, -half, half, 0.0, nz * cell, 1.0, 12000, 3,
                    nx=nx, ny=ny, nz=nz, ox=-half, oy=-half, oz=0.0, cell=cell, material=material, field=fld,
                    field_mode=field_mode)
    mu = spectrum_muons(3, n, "square")
    if half < 1.0:                       # shrunken test grid: keep the start square inside it
        mu.pos_q[:, :2] *= np.float32(half)
    return Workload("config3_field_map_shield", hist, geom, mu, seed=1)


CONFIG4_TABLE_SHAPES = [(50, 128, 64), (100, 256, 128), (256, 1024, 512)]
