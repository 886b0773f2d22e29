"""bench.py — throughput of the muon-transport hot path (BASELINE.json metric: muon-steps/s and muons/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--muons M]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one mt_transport call: the whole hot path over one batch of synthetic
muons of BASELINE.json configs[3] (10^7 muons, 200x200x3000 voxel field map) — the config north_star's
roofline target is quoted on.  Rank r transports its own 10^7 muons (ids r*M ..), no collective on the data
path (weak scaling).  One JSON line on stdout (rank 0); everything else goes to stderr.

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
`--sweep` runs BASELINE.json configs[4] instead (10^8 muons in batches of 10^7 at each table shape and placement — with
`--gpus N` batch k on rank k % N — then, on one GPU, muons-per-launch 2^14 .. 2^24) and prints one JSON line per point.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# algorithmic thread-operations and gathered bytes per muon-step (contract operations of
# DESIGN.md §3 counted one each; loads not counted as operations)
ALG_OPS_PER_STEP = {"voxel": 383, "regions": 308, "poly": 349}
ALG_GATHER_BYTES_PER_STEP = {"voxel": 168, "regions": 40, "poly": 50}


def variant_work(mode, field_mode=0, joint=False):
    """(ops, gathered bytes) per muon-step of a SURVEY.md §8(f) variant, by the counting rules of DESIGN.md §7:
    nearest-neighbour field = no trilinear (78 ops, 128 B) but one 16-byte cell record; field at every RK4 stage = three
    more stage positions (3 fma), lookups (voxel: 12 for the cell and the inside test + the interpolation; regions: 20;
    polyhedra: 61) and c1 * B products (3); joint tables = one draw instead of two, an integer cell split, no polar
    sine / cosine, one more square root."""
    ops, gb = ALG_OPS_PER_STEP[mode], ALG_GATHER_BYTES_PER_STEP[mode]
    interp_ops, interp_b = (78, 128) if mode == "voxel" else (0, 0)
    if mode == "voxel" and (field_mode & 1):
        ops, gb = ops - 78 + 1, gb - 128 + 16
        interp_ops, interp_b = 6, 16
    if field_mode & 2:
        lookup = {"voxel": 12 + interp_ops, "regions": 20, "poly": 61}[mode]
        ops, gb = ops + 2 + 3 * (3 + lookup + 3), gb + 3 * (interp_b if mode == "voxel" else 0)
    if joint:
        ops += -6 + 3 - 23 + 8
    return ops, gb
# Work the host and the grid repack do once, which the counting rules above still charge to every step: the 18 Philox
# round-key increments (host-made, every mode) and the 12 x-differences of the trilinear corners (stored in the repacked
# grid).  `frac` is quoted on the full algorithmic count; `frac_without_precomputed` on the count minus these.
PRECOMPUTED_OPS = {"philox_round_keys": 18, "trilinear_x_differences": 12}

# The ncu launch list of one timed step (per-launch time, DRAM bytes, L2 bytes, L1 sectors, L1 data-stage wavefronts,
# warp instructions), committed as text; profiles/r3_launches.md names the command.  bench.py cannot run ncu itself: it
# READS this file, and uses it only for a run of the very configuration it was captured on — anything else gets null.
NCU_LAUNCH_LIST = "profiles/r3_launches.csv"
NCU_CAPTURE_CONFIG = dict(config=3, muons=10_000_000, field_mode=0, joint=False, poly=False, sched=0, placement=0, block=0,
                          slab=0, lanes=0, sort_every=0, pass_mode=0, no_lean=False, blocks_per_sm=0, min_idle=0,
                          draws=1_000_000, n_cells=8, half_width_cells=100)


def ncu_capture(args):
    """Sums over the launches of each kernel in NCU_LAUNCH_LIST, or None if this run is not the captured configuration
    (or the file is missing / unreadable)."""
    if any(getattr(args, k) != v for k, v in NCU_CAPTURE_CONFIG.items()):
        return None
    import csv
    try:
        with open(os.path.join(ROOT, NCU_LAUNCH_LIST), newline="") as f:
            rows = list(csv.DictReader(f))
    except OSError:
        return None
    agg = {}
    for r in rows:
        name = r["kernel"].replace("void ", "").split("<")[0].split("(")[0]
        a = agg.setdefault(name, {"launches": 0})
        a["launches"] += 1
        for k, v in r.items():
            if k.endswith(".sum") and v != "":
                a[k] = a.get(k, 0.0) + float(v)
    return agg or None


SM_COUNT, LANES_PER_SM = 148, 128          # B200: 4 SMSPs x 32 lanes issue one warp instruction per clock


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu, self.rows, self.proc, self.thread = gpu_index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return self
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()
        return self

    def _read(self):
        for line in self.proc.stdout:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) >= 9:
                self.rows.append(parts)

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"], samples=0)
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=5)
        sm, mx, reasons, power = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); power.append(float(r[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm), power_w_max=max(power) if power else None)


# ------------------------------------------------------------------------------------------ roofline
def roofline_block(mode, steps_per_call, t_call_s, launches_per_step, lanes, n_muons, grid_bytes, peaks, mp, field_mode=0,
                   joint=False, capture=None, probe_clocks=None):
    """north_star's roofline for one step of this rank: "the larger of FP32-issue time ... at peak and gather bytes at
    L2/HBM bandwidth".  Every term that can be evaluated for this run is evaluated, `bound` is the LARGEST of them, and
    `achieved` / `peak` / `frac` are that term's.  Terms:
      alu            algorithmic thread-operations at the nominal issue peak, one per lane per clock — the
                     peak DESIGN.md derives from unit counts and the measured sm_max_mhz; `frac_nominal` is this term's
                     fraction whatever binds (the figure comparable across rounds)
      hbm            compulsory HBM bytes (muon state in and out + the field grid once) at the measured copy bandwidth
      l1 / l2 / dram L1 data-stage wavefronts at one per SM per clock, L2 bytes at the L2 random-sector rate measured in
                     this process, DRAM bytes at the measured copy bandwidth — MEASURED traffic of the dominant kernel from
                     the committed ncu launch list, only when this run is the configuration that list was captured on
    mp: mt_measure_peaks of this process, or None if the probe failed (then only nominal / driver-measured peaks are used).
    The per-lane gather estimate (every lane's record a sector of its own) is printed as an upper estimate and takes no
    part in `bound`: lanes of a sorted warp share sectors."""
    ops_step, gb_step = variant_work(mode, field_mode, joint)
    pre = PRECOMPUTED_OPS["philox_round_keys"] + (PRECOMPUTED_OPS["trilinear_x_differences"]
                                                  if mode == "voxel" and not (field_mode & 1) else 0)
    ops = steps_per_call * ops_step                                        # thread-operations per step
    gbytes = steps_per_call * gb_step                                      # gathered bytes per step, one sector per lane
    clock_hz = peaks["sm_max_mhz"] * 1e6
    nominal = SM_COUNT * LANES_PER_SM * clock_hz                           # thread-ops/s: one per lane per clock
    hbm_bps = peaks["hbm_gbs"] * 1e9
    per_lane = launches_per_step // max(lanes, 1)
    passes = lanes * ((per_lane - 3) // 3 + 1 if per_lane > 3 else per_lane)      # launches of the transport kernel
    state_bytes = 64 * n_muons + grid_bytes                                # compulsory HBM traffic
    dominant = "wave_transport_kernel" if per_lane > 1 else "transport_kernel"
    cap = (capture or {}).get(dominant)
    if cap and cap["launches"] != passes:
        cap = None                                                         # not the launch sequence that was captured

    # ---- the terms (seconds per step), each with what was achieved and the peak it is held against
    terms = {"alu": dict(t=ops / nominal, achieved=ops / t_call_s / 1e12, peak=nominal / 1e12, unit="T thread-ops/s",
                         basis="algorithmic ops, nominal issue peak 148 SM x 128 lanes x sm_max_mhz"),
             "hbm": dict(t=state_bytes / hbm_bps, achieved=state_bytes / t_call_s / 1e9, peak=peaks["hbm_gbs"], unit="GB/s",
                         basis="compulsory bytes, %s copy bandwidth" % peaks["source"])}
    if cap:
        wf = cap.get("l1tex__data_pipe_lsu_wavefronts.sum")
        if wf:
            terms["l1"] = dict(t=wf / (SM_COUNT * clock_hz), achieved=wf / t_call_s / 1e9, peak=SM_COUNT * clock_hz / 1e9,
                               unit="G wavefronts/s", basis="measured L1 data-stage wavefronts (ncu), one per SM per clock")
        l2b = cap.get("lts__t_bytes.sum")
        if l2b and mp:
            terms["l2"] = dict(t=l2b / mp["gather_64m_bytes_per_s"], achieved=l2b / t_call_s / 1e9,
                               peak=mp["gather_64m_bytes_per_s"] / 1e9, unit="GB/s",
                               basis="measured L2 bytes (ncu), random-sector L2 rate measured in this process")
        db = cap.get("dram__bytes_read.sum", 0.0) + cap.get("dram__bytes_write.sum", 0.0)
        if db:
            terms["dram"] = dict(t=db / hbm_bps, achieved=db / t_call_s / 1e9, peak=peaks["hbm_gbs"], unit="GB/s",
                                 basis="measured DRAM bytes (ncu), %s copy bandwidth" % peaks["source"])
    bound = max(terms, key=lambda k: terms[k]["t"])
    top = terms[bound]
    frac = top["t"] / t_call_s
    ranked = sorted(terms, key=lambda k: -terms[k]["t"])
    reading = "largest term: %s, %.1f of %.1f ms measured (%.2f); then %s" % (
        bound, 1e3 * top["t"], 1e3 * t_call_s, frac,
        ", ".join("%s %.1f ms" % (k, 1e3 * terms[k]["t"]) for k in ranked[1:]))
    if frac < 0.5:
        reading += ("; no throughput term reaches half of the measured time: with %d muons on %d SMs the call is bound by the "
                    "latency of one history's dependent steps and by the tails of its launches, not by a unit" % (n_muons, SM_COUNT))
    if not cap:
        reading += "; no ncu capture of this configuration: the l1 / l2 / dram terms are not evaluated"
    dram = terms["dram"]["t"] * hbm_bps if "dram" in terms else None
    out = {
        "bound": bound, "unit": top["unit"], "achieved": top["achieved"], "peak": top["peak"], "frac": frac,
        "peak_source": top["basis"],
        "frac_nominal": terms["alu"]["t"] / t_call_s, "peak_nominal": nominal / 1e12,
        "frac_nominal_is": "algorithmic thread-ops (%d per muon-step) over the nominal issue peak; the same figure as "
                           "BENCH_r01 / r02's frac_nominal" % ops_step,
        "frac_without_precomputed": (ops_step - pre) / ops_step * terms["alu"]["t"] / t_call_s,
        "ops_per_muon_step": ops_step, "ops_per_muon_step_without_precomputed": ops_step - pre,
        "gather_bytes_per_muon_step": gb_step,
        "kernel": ("wave_transport_kernel: %d z-slab passes (%d lane(s)) among the %d launches of a step (the rest sort "
                   "the live list)" % (passes, lanes, launches_per_step)) if per_lane > 1 else
                  "transport_kernel (%d launch(es) per step)" % launches_per_step,
        "terms_ms": dict({"measured": 1e3 * t_call_s}, **{k: 1e3 * v["t"] for k, v in terms.items()}),
        "terms_basis": {k: v["basis"] for k, v in terms.items()},
        "reading": reading,
        "ncu_capture": NCU_LAUNCH_LIST if cap else None,
        "traffic": (dram / passes) if dram else None,
        "traffic_unit": "DRAM bytes per launch of the kernel = per-step total / passes (ncu launch list)",
        "traffic_per_batch": dram,
        "algorithmic_hbm_bytes_per_batch": state_bytes,
        "algorithmic_hbm_bytes_note": "64 B of state per muon + the library's 32-byte-per-cell field grid read once",
        "traffic_over_algorithmic": (dram / state_bytes) if dram else None,
    }
    if cap:
        steps32 = steps_per_call / 32.0
        out["measured_per_warp_step"] = {
            "basis": "ncu launch list / (muon-steps / 32); a warp-step here is 32 muon-steps, whatever the lanes' activity",
            "l1_wavefronts": cap.get("l1tex__data_pipe_lsu_wavefronts.sum", 0.0) / steps32,
            "l1_sectors": cap.get("l1tex__t_sectors.sum", 0.0) / steps32,
            "l2_sectors": cap.get("lts__t_sectors.sum", 0.0) / steps32,
            "warp_instructions": cap.get("smsp__inst_executed.sum", 0.0) / steps32,
            "by_source": "profiles/r3_l1_sources.md"}
    if mp:
        measured = mp["ffma_thread_ops_per_s"]                             # a pure FFMA stream on this device, now
        out["frac_measured"] = ops / measured / t_call_s
        out["peak_measured"] = measured / 1e12
        out["peak_measured_source"] = ("mt_measure_peaks in this process after the timed region: fma.rn.f32 stream, 8 warps "
                                       "per scheduler; SM clock while it ran: %s"
                                       % (probe_clocks if probe_clocks is not None else "not sampled"))
        out["gather_one_sector_per_lane_upper_ms"] = {
            "note": "every lane's record priced as a 32-byte sector of its own at that level's random-sector rate; an upper "
                    "estimate that takes no part in `bound`",
            "l1_resident_64k": 1e3 * gbytes / mp["gather_l1_bytes_per_s"],
            "l2_resident_64m": 1e3 * gbytes / mp["gather_64m_bytes_per_s"],
            "hbm_1400m": 1e3 * gbytes / mp["gather_1400m_bytes_per_s"]}
        out["measured_peaks"] = {
            "ffma_T_thread_ops_per_s": measured / 1e12, "lop3_T": mp["lop3_thread_ops_per_s"] / 1e12,
            "imad_T": mp["imad_thread_ops_per_s"] / 1e12, "mulhi_T": mp["mulhi_thread_ops_per_s"] / 1e12,
            "mufu_T": mp["mufu_thread_ops_per_s"] / 1e12,
            # mixed streams as a fraction of the fma rate: near 1 = that pipe runs beside the FP32 stream,
            # 0.75 / 0.625 = its instructions take 2 / 4 FP32 issue cycles each
            "mix_over_ffma": {"8_fma_4_lop3": mp["mix_ffma8_lop3_4_thread_ops_per_s"] / measured,
                              "8_fma_4_imad": mp["mix_ffma8_imad4_thread_ops_per_s"] / measured,
                              "8_fma_2_mulwide": mp["mix_ffma8_mulwide2_thread_ops_per_s"] / measured},
            "gather_TB_per_s": {"l1_resident_64k": mp["gather_l1_bytes_per_s"] / 1e12,
                                "l2_resident_675k": mp["gather_675k_bytes_per_s"] / 1e12,
                                "l2_resident_64m": mp["gather_64m_bytes_per_s"] / 1e12,
                                "hbm_1400m": mp["gather_1400m_bytes_per_s"] / 1e12},
            "hbm_copy_gbs_%s" % peaks["source"]: peaks["hbm_gbs"]}
    else:
        out["measured_peaks"] = None
        out["measured_peaks_note"] = "mt_measure_peaks failed in this process: nominal and driver-measured peaks only"
    return out


# ------------------------------------------------------------------------------------------ workload
def make_workload(config, n_muons, device, rank, joint=False, field_mode=0, poly=False, n_draws=1_000_000, n_cells=8,
                  half_width_cells=100):
    """BASELINE.json configs[config] with this rank's batch of muons (generator batch = rank).  n_cells / half_width_cells:
    config 3 on another voxel grid (3.75 m of z per shield cell at 1 cm, 2 x half_width_cells cells across; the defaults
    are configs[3]'s 200x200x3000) — profiles/r3_slab_grids.md."""
    from paper_2512_10520_b200 import workloads as w
    t0 = time.time()
    if config == 3:
        wl = w.config3(n=8, device=device, joint=joint, field_mode=field_mode, n_draws=n_draws, n_cells=n_cells,
                       half_width_cells=half_width_cells)                # histograms + voxel grids (made on the GPU)
        wl.muons = w.spectrum_muons(3, n_muons, "square", batch=rank)
        if half_width_cells < 100:                                        # a grid narrower than the 2 m start square
            wl.muons.pos_q[:, :2] *= np.float32(half_width_cells * 0.01)
    elif config == 2:
        # --poly: config 2's muons and tables in the tapered-magnet polyhedra geometry
        wl = w.config2p(n=8, joint=joint, n_draws=n_draws) if poly else w.config2(n=8, joint=joint, n_draws=n_draws)
        wl.geom.field_mode = field_mode & 2
        wl.muons = w.spectrum_muons(2, n_muons, "square", batch=rank)
    elif config == 1:
        wl = w.config1(n=8, joint=joint, n_draws=n_draws)
        wl.geom.field_mode = field_mode & 2
        wl.muons = w.spectrum_muons(1, n_muons, "gauss", batch=rank)
    elif config == 0:
        # the oracle-sized parity case (4096 identical muons by default): timed only to fill BASELINE.md's table
        wl = w.config0(n=n_muons, joint=joint, n_draws=n_draws)
    else:
        raise SystemExit("bench.py times BASELINE.json configs 0-3; configs[4] is --sweep")
    log("[bench] rank %d: %s, %d muons generated in %.1f s" % (rank, wl.name, n_muons, time.time() - t0))
    return wl


def oracle_sample(wl, n_muons, id_base, target_seconds, threads=None):
    """Time the CPU oracle (as it stands) on an id-strided sample of this workload sized to ~target_seconds.
    Returns (muon-steps/s, muons/s, cores, description, runner) where runner() repeats the sized sample."""
    import oracle
    threads = threads or oracle.max_threads()
    T, G = oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom)

    def run(sel):
        t0 = time.perf_counter()
        r = oracle.transport(T, G, wl.muons.pos_q[sel], wl.muons.mom[sel], wl.seed, ids=(id_base + sel).astype(np.uint64),
                             threads=threads)
        return time.perf_counter() - t0, int(r["steps"].sum()), len(sel)

    pilot = np.arange(0, n_muons, max(1, n_muons // 2048), dtype=np.int64)[:2048]
    dt, steps, _ = run(pilot)
    rate = steps / max(dt, 1e-9)
    per_muon = steps / max(len(pilot), 1)
    n_sample = int(min(n_muons, max(len(pilot), target_seconds * rate / max(per_muon, 1.0))))
    sel = np.arange(0, n_muons, max(1, n_muons // n_sample), dtype=np.int64)[:n_sample]
    desc = "every %dth muon of the batch (%d muons), float32 contract mode, OpenMP over muons" % (max(1, n_muons // n_sample), len(sel))
    return threads, desc, (lambda: run(sel))


# --------------------------------------------------------------------------------------- reference arm
def run_reference(args, rank, world):
    """The CPU oracle on host cores, same config / metric / unit; rank 0 alone works and prints, the other ranks only
    join the (gloo) process group so that the line's n_gpus is the number of ranks that really ran."""
    dist, joined = join_ranks(args, rank, world, 0, "gloo")
    if rank != 0:
        dist.barrier()
        dist.destroy_process_group()
        return
    import torch
    dev = "cuda" if torch.cuda.is_available() else "cpu"          # the grid generator may use the GPU; the timed code never does
    wl = make_workload(args.config, args.muons, dev, 0, args.joint, args.field_mode, args.poly, args.draws, args.n_cells,
                       args.half_width_cells)
    cores, desc, runner = oracle_sample(wl, args.muons, 0, args.ref_seconds, threads=args.ref_threads or None)
    for _ in range(args.warmup):
        runner()
    t_tot, s_tot, m_tot = 0.0, 0, 0
    for _ in range(args.steps):
        dt, s, m = runner()
        t_tot += dt; s_tot += s; m_tot += m
    value = s_tot / t_tot
    line = {
        "impl": "reference", "metric": "muon_steps_per_s", "value": value, "unit": "muon-steps/s",
        "muons_per_s": m_tot / t_tot, "n_gpus": joined, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_tot / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": wl.name, "muons_per_step": m_tot // max(args.steps, 1), "sample": desc},
        "cpu_baseline": {"value": value, "unit": "muon-steps/s", "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": "muon-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------- our arm
def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2512_10520_b200 import binding as b, build as lib_build

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the transport path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if rank == 0:
        lib_build.build()
    _, joined = join_ranks(args, rank, world, local_rank, "nccl")
    if world > 1:
        dist.barrier()
    b.lib()

    from paper_2512_10520_b200.sharding import gather_ranges, reduce_job, weak_shard
    shard = weak_shard(args.muons, rank, world)               # own batch, own id range, no collective
    n, id_base = shard.n, shard.id_base
    wl = make_workload(args.config, n, dev, rank, args.joint, args.field_mode, args.poly, args.draws, args.n_cells,
                       args.half_width_cells)
    mode = {0: "regions", 1: "voxel", 2: "poly"}[wl.geom.mode]
    grid_bytes = 32 * (wl.geom.nx + 2) * (wl.geom.ny + 2) * (wl.geom.nz + 2) if mode == "voxel" else 0
    h = b.MuonTransport(local_rank).setup(wl.hist, wl.geom, args.placement)
    h.set_option(b.MT_OPT_SCHEDULE, args.sched).set_option(b.MT_OPT_BLOCK_THREADS, args.block)
    h.set_option(b.MT_OPT_SLAB_CELLS, args.slab).set_option(b.MT_OPT_REFILL_MIN_IDLE, args.min_idle)
    h.set_option(b.MT_OPT_BLOCKS_PER_SM, args.blocks_per_sm).set_option(b.MT_OPT_NO_LEAN, int(args.no_lean))
    h.set_option(b.MT_OPT_LANES, args.lanes).set_option(b.MT_OPT_PASS_MODE, args.pass_mode)
    h.set_option(b.MT_OPT_SORT_EVERY, args.sort_every)
    host_geom = None
    if rank == 0 and not args.no_cpu_baseline:
        import copy
        host_geom = copy.copy(wl.geom)                       # host copies for the oracle, made before the grids are freed
        if mode == "voxel":
            host_geom.material, host_geom.field = wl.geom.material.cpu().numpy(), wl.geom.field.cpu().numpy()
    wl.geom.material = wl.geom.field = None                   # the library repacked them; free 1.5 GB
    torch.cuda.empty_cache()

    stream = torch.cuda.Stream(device=dev)
    d_pos, d_mom = torch.from_numpy(wl.muons.pos_q).to(dev), torch.from_numpy(wl.muons.mom).to(dev)
    out = {"pos_flag": torch.empty((n, 4), dtype=torch.float32, device=dev),
           "mom_steps": torch.empty((n, 4), dtype=torch.float32, device=dev)}
    torch.cuda.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident leg: inputs already in HBM; CUDA events on the launching stream around every step
    def one_step():
        return h.transport(d_pos, d_mom, wl.seed, id_base=id_base, out=out, stream=stream)

    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            res = one_step()
        stream.synchronize()
        steps_per_call = int(res["counters"][0].item())
        barrier()
        sampler = ClockSampler(local_rank).start() if rank == 0 else None
        launches0 = b.mt_launch_count(h.ctx)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        wall0 = time.perf_counter()
        for e0, e1 in evs:
            e0.record(stream)
            one_step()
            e1.record(stream)
        stream.synchronize()
        barrier()
        wall = time.perf_counter() - wall0
        clocks = sampler.stop() if sampler else None
        launches = b.mt_launch_count(h.ctx) - launches0
        lanes_used = b.mt_get_info(h.ctx, b.MT_INFO_LAST_LANES)
    dev_ms = [e0.elapsed_time(e1) for e0, e1 in evs]
    t_dev = sum(dev_ms) * 1e-3
    flags = np.bincount(out["pos_flag"][:, 3].view(torch.int32).cpu().numpy(), minlength=5)[1:5]

    # ---- end-to-end leg: HOST (pinned) buffers through mt_transport_host, copies inside the timed region
    pin = lambda a: torch.from_numpy(a).pin_memory()
    h_pos, h_mom = pin(wl.muons.pos_q), pin(wl.muons.mom)
    h_out = {"pos_flag": torch.empty((n, 4), dtype=torch.float32).pin_memory(),
             "mom_steps": torch.empty((n, 4), dtype=torch.float32).pin_memory()}
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    h.transport_host(h_pos, h_mom, wl.seed, id_base=id_base, out=h_out, stream=stream)      # warm-up: staging buffers
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        r = h.transport_host(h_pos, h_mom, wl.seed, id_base=id_base, out=h_out, stream=stream)
    barrier()
    t_e2e = time.perf_counter() - t0
    assert int(r["counters"][0]) == steps_per_call
    h2d = h_pos.numel() * 4 + h_mom.numel() * 4
    d2h = h_out["pos_flag"].numel() * 4 + h_out["mom_steps"].numel() * 4 + 64

    # ---- max over ranks, totals over ranks
    (t_dev_max, t_e2e_max, wall_max), (steps_all, muons_all) = reduce_job(
        [t_dev, t_e2e, wall], [steps_per_call, n], dist if world > 1 else None, dev)
    id_ranges = gather_ranges(shard, dist if world > 1 else None, dev)
    h.close()
    if rank != 0:
        return

    peaks = load_peaks()
    value = steps_all * args.steps / t_dev_max
    e2e_value = steps_all * e2e_steps / t_e2e_max
    # The probe runs after the timed region (1.4 GB of its own, ~50 ms): a failure there must not cost the line, and the
    # clock it ran at is recorded beside the peak it gives
    mp, probe_clocks = None, None
    try:
        probe_sampler = ClockSampler(local_rank).start()
        for _ in range(3):                                    # (long enough for a few 100 ms clock samples)
            mp = b.mt_measure_peaks(local_rank)
        probe_clocks = probe_sampler.stop().get("sm_mhz")
    except Exception as e:                                    # MtError, OSError from nvidia-smi, ...
        log("[bench] peak probe failed (%s): nominal peaks only" % e)
    roofline = roofline_block(mode, steps_per_call, t_dev / args.steps, max(1, launches // args.steps), lanes_used, n,
                              grid_bytes, peaks, mp, args.field_mode, args.joint, ncu_capture(args), probe_clocks)
    line = {
        "metric": "muon_steps_per_s", "value": value, "unit": "muon-steps/s",
        "muons_per_s": muons_all * args.steps / t_dev_max,
        "n_gpus": joined, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_dev_max / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": wl.name + ("+joint2d" if args.joint else "") + ("+field_mode%d" % args.field_mode if args.field_mode else ""),
                   "muons_per_gpu": n, "muon_steps_per_gpu_step": steps_per_call,
                   "schedule": args.sched, "placement": args.placement, "block": args.block, "slab_cells": args.slab,
                   "lanes": lanes_used,
                   "parallelism": "id-range sharding x%d, replicated tables and grids, no collective" % world,
                   "id_ranges": id_ranges,
                   "l2": "inputs larger than L2 (%d MB muon state in + out, %d MB field grid per step)" % (64 * n // 10 ** 6, grid_bytes // 10 ** 6),
                   "grid": [wl.geom.nx, wl.geom.ny, wl.geom.nz] if mode == "voxel" else None,
                   "flags_rank0": {"stopped": int(flags[0]), "exited": int(flags[1]), "escaped": int(flags[2]),
                                   "maxsteps": int(flags[3])}},
        "e2e": {"value": e2e_value, "unit": "muon-steps/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "ms_per_step": 1e3 * t_e2e_max / e2e_steps},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": roofline,
        "wall_ms_per_step": 1e3 * wall_max / args.steps,
        "dev_ms_steps": [round(x, 3) for x in dev_ms],
    }
    if host_geom is not None:
        wl.geom = host_geom
        cores, desc, runner = oracle_sample(wl, n, id_base, args.ref_seconds)
        dt, s, m = runner()
        line["cpu_baseline"] = {"value": s / dt, "unit": "muon-steps/s", "cores": cores, "kind": "oracle",
                                "sample": desc, "muons_per_s": m / dt, "seconds": dt}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------ configs[4] sweep
def run_sweep(args, rank, world, local_rank):
    """BASELINE.json configs[4]: (A) 10^8 muons in 10 batches of 10^7 (id_base = batch * 10^7) for every table shape x
    placement — with N ranks, batch k runs on rank k % N (sharding.batch_shard; replicated tables and grids, no collective
    on the data path), a point's time is the MAX over ranks of each rank's summed device time and its muon-steps the SUM;
    (B) muons per launch 2^14 .. 2^24 on the middle shape, one GPU by nature (rank 0 of a 1-rank job only).  One JSON line
    per point, printed by rank 0."""
    import torch
    import torch.distributed as dist
    from paper_2512_10520_b200 import binding as b, build as lib_build, workloads as w
    from paper_2512_10520_b200.sharding import batch_shard, reduce_job
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the transport path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if rank == 0:
        lib_build.build()
    _, joined = join_ranks(args, rank, world, local_rank, "nccl")
    if world > 1:
        dist.barrier()
    job = dist if world > 1 else None
    peaks = load_peaks()
    alu_peak = joined * SM_COUNT * LANES_PER_SM * peaks["sm_max_mhz"] * 1e6
    n_batch, n_batches = args.muons, args.sweep_batches
    mine = batch_shard(n_batches, rank, world)
    stream = torch.cuda.Stream(device=dev)
    base = w.config3(n=8, device=dev)                        # grids once; histograms are regenerated per shape
    n_launch_max = 1 << 24                                   # part (B)'s largest launch
    n_out = max(n_batch, n_launch_max) if world == 1 else n_batch
    out = {"pos_flag": torch.empty((n_out, 4), dtype=torch.float32, device=dev),
           "mom_steps": torch.empty((n_out, 4), dtype=torch.float32, device=dev)}

    def timed(h, d_pos, d_mom, id_base, o):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            e0.record(stream)
            r = h.transport(d_pos, d_mom, base.seed, id_base=id_base, out=o, stream=stream)
            e1.record(stream)
            stream.synchronize()
        return e0.elapsed_time(e1) * 1e-3, int(r["counters"][0].item())

    def emit(**kw):
        if rank != 0:
            return
        kw["n_gpus"] = joined
        kw["roofline_frac_nominal"] = kw["muon_steps_per_s"] * ALG_OPS_PER_STEP["voxel"] / alu_peak
        print(json.dumps(kw), flush=True)

    batches = {k: w.spectrum_muons(3, n_batch, "square", batch=k) for k in mine}
    o_batch = {k: v[:n_batch] for k, v in out.items()}
    for shape in w.CONFIG4_TABLE_SHAPES:
        t0 = time.time()
        hist = w.shield_histograms(3, [1.0, 1.0, 10.0], shape[0], shape[1], shape[2], args.sweep_draws)
        log("[sweep] rank %d: tables %dx%dx%d generated in %.1f s" % ((rank,) + shape + (time.time() - t0,)))
        for placement, pname in ((b.MT_PLACE_AUTO, "auto"), (b.MT_PLACE_L2, "l2"), (b.MT_PLACE_SMEM, "smem")):
            h = b.MuonTransport(local_rank)
            try:
                h.setup(hist, base.geom, placement)
                h.set_option(b.MT_OPT_SCHEDULE, args.sched)
                if mine:
                    k0 = mine[0]
                    d0, m0 = torch.from_numpy(batches[k0].pos_q).to(dev), torch.from_numpy(batches[k0].mom).to(dev)
                    for _ in range(2):
                        timed(h, d0, m0, k0 * n_batch, o_batch)      # warm-up
                if world > 1:
                    torch.cuda.synchronize()
                    dist.barrier()
                t_tot, s_tot = 0.0, 0
                for k in mine:                                   # batch k of the job: generator batch k, ids from k * n_batch
                    d_pos, d_mom = torch.from_numpy(batches[k].pos_q).to(dev), torch.from_numpy(batches[k].mom).to(dev)
                    dt, st = timed(h, d_pos, d_mom, k * n_batch, o_batch)
                    t_tot += dt; s_tot += st
                (t_max,), (s_all, m_all, b_all) = reduce_job([t_tot], [s_tot, n_batch * len(mine), len(mine)], job, dev)
                emit(sweep="table_shape", pbins_x_dp_x_theta="%dx%dx%d" % shape, placement=pname,
                     muons=int(m_all), batches=int(b_all), batches_by_rank="batch k on rank k %% %d" % world,
                     muon_steps=int(s_all), seconds=t_max, muon_steps_per_s=s_all / t_max, muons_per_s=m_all / t_max)
            except b.MtError as e:                               # (the same refusal on every rank: no reduction to match)
                emit(sweep="table_shape", pbins_x_dp_x_theta="%dx%dx%d" % shape, placement=pname,
                     muon_steps_per_s=0.0, unsupported=str(e))
            finally:
                h.close()
        if shape == w.CONFIG4_TABLE_SHAPES[1] and world == 1:
            h = b.MuonTransport(local_rank).setup(hist, base.geom, b.MT_PLACE_AUTO)
            h.set_option(b.MT_OPT_SCHEDULE, args.sched)
            mu = w.spectrum_muons(3, n_launch_max, "square", batch=0)     # 2^24 muons of their own: the last point is a real
            d_pos, d_mom = torch.from_numpy(mu.pos_q).to(dev), torch.from_numpy(mu.mom).to(dev)      # 16 777 216-muon call
            for log2n in range(14, 25, 2):
                n = 1 << log2n
                o = {"pos_flag": out["pos_flag"][:n], "mom_steps": out["mom_steps"][:n]}
                best, st = None, 0
                for rep in range(4):
                    dt, st = timed(h, d_pos[:n], d_mom[:n], 0, o)
                    best = dt if best is None or (rep > 0 and dt < best) else best
                emit(sweep="muons_per_launch", pbins_x_dp_x_theta="%dx%dx%d" % shape, placement="auto", muons=n,
                     muon_steps=st, seconds=best, muon_steps_per_s=st / best, muons_per_s=n / best)
            h.close()
            del d_pos, d_mom, mu
    if world > 1:
        torch.cuda.synchronize()
        dist.barrier()
        dist.destroy_process_group()


def self_launch(n_gpus):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start the N ranks ourselves, one process per
    GPU, exactly as the driver's own command line would (torch.distributed.run, 127.0.0.1 rendezvous), and pass the
    ranks' output through.  Rank 0 prints the JSON line."""
    import socket
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    env = dict(os.environ)
    # leave the communicator log on (the ranks that joined can be counted from it) but keep stdout to the one JSON line
    env.setdefault("NCCL_DEBUG", "INFO")
    env.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
    env["MT_BENCH_SELF_LAUNCHED"] = "1"
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n_gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    log("[bench] --gpus %d without a torchrun environment: launching %s" % (n_gpus, " ".join(cmd)))
    raise SystemExit(subprocess.call(cmd, env=env))


def join_ranks(args, rank, world, local_rank, backend):
    """Process group of the job; returns (dist or None, ranks that actually joined).  The line's n_gpus is that count,
    and a count that differs from --gpus is refused rather than printed."""
    if world == 1:
        return None, 1
    import torch
    import torch.distributed as dist
    if backend == "nccl":
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        one = torch.ones(1, dtype=torch.int64, device=torch.device("cuda", local_rank))
    else:
        dist.init_process_group("gloo")
        one = torch.ones(1, dtype=torch.int64)
    dist.all_reduce(one)
    joined = int(one.item())
    if joined != args.gpus:
        raise SystemExit("bench.py: --gpus %d but %d ranks joined the process group" % (args.gpus, joined))
    return dist, joined


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--muons", type=int, default=10_000_000, help="muons per GPU per step")
    ap.add_argument("--sched", type=int, default=0, help="MT_SCHED_* (0 = library default)")
    ap.add_argument("--placement", type=int, default=0, help="MT_PLACE_* (0 = auto)")
    ap.add_argument("--block", type=int, default=0)
    ap.add_argument("--blocks-per-sm", type=int, default=0)
    ap.add_argument("--slab", type=int, default=0)
    ap.add_argument("--min-idle", type=int, default=0)
    ap.add_argument("--lanes", type=int, default=0, help="MT_OPT_LANES: concurrent lanes per call (0 = library default)")
    ap.add_argument("--sort-every", type=int, default=0, help="MT_OPT_SORT_EVERY: re-sort the live list after every k-th pass")
    ap.add_argument("--pass-mode", type=int, default=0, help="MT_OPT_PASS_MODE: 1 persistent CTAs, 2 one item per warp (0 = default)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--ref-seconds", type=float, default=15.0, help="CPU work per oracle sample")
    ap.add_argument("--ref-threads", type=int, default=0, help="--impl reference: oracle threads (0 = all host cores)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--joint", action="store_true", help="the paper's joint 2D histograms (DESIGN.md 3.10) instead of two 1D ones")
    ap.add_argument("--field-mode", type=int, default=0, help="MT_FIELD_*: 1 nearest, 2 per-stage, 3 both (DESIGN.md 3.11)")
    ap.add_argument("--no-lean", action="store_true", help="MT_OPT_NO_LEAN: general kernels even where the lean variant applies")
    ap.add_argument("--poly", action="store_true", help="with --config 2: the convex-polyhedra shield (DESIGN.md 3.12)")
    ap.add_argument("--n-cells", type=int, default=8, help="config 3: shield cells along z, 375 grid layers each (8 = configs[3])")
    ap.add_argument("--half-width-cells", type=int, default=100, help="config 3: half the grid's width in cells (100 = configs[3])")
    ap.add_argument("--sweep", action="store_true", help="BASELINE.json configs[4] (table shapes, muons per launch)")
    ap.add_argument("--probes", action="store_true", help="only the in-process peak and field-path probes (one JSON line)")
    ap.add_argument("--draws", type=int, default=1_000_000, help="draws per generated histogram (BASELINE.json: 10^6)")
    ap.add_argument("--sweep-batches", type=int, default=10)
    ap.add_argument("--sweep-draws", type=int, default=1_000_000, help="draws per generated histogram")
    args = ap.parse_args()
    if args.warmup < 1:
        args.warmup = 1
    if args.probes:
        from paper_2512_10520_b200 import binding as b, build as lib_build
        lib_build.build()
        fp = b.mt_probe_field_paths(0)
        print(json.dumps({"measured_peaks": b.mt_measure_peaks(0),
                          "field_paths_TB_per_s": {k[:3]: v * 32 / 1e12 for k, v in fp.items() if k.endswith("_per_s")},
                          "field_paths_records_per_launch": fp["records_per_launch"]}), flush=True)
        return
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be at least 1")
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        self_launch(args.gpus)                                   # does not return
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        # one rank per GPU or nothing: a line that says n_gpus = N must come from N ranks
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d (launch with --nproc-per-node %d, or drop the torchrun "
                         "environment and let bench.py start the ranks)" % (args.gpus, world, args.gpus))
    # every rank generates its own inputs: share the host cores instead of fighting for them
    os.environ.setdefault("MT_GEN_WORKERS", str(max(1, (os.cpu_count() or 1) // max(world, 1))))
    if args.sweep:
        run_sweep(args, rank, world, local_rank)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
