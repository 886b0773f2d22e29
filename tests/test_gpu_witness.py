"""-m gpu: the CUDA path against the oracle's libm witness at north_star's REAL tolerance (VERDICT r1 next #1c).

Every other parity test compares with the contract-mode oracle and therefore reads "100 % bit-exact"; here the
reference is the oracle run with the C library's exp2 / sin / cos (oracle `libm=True`), i.e. the plain definitions the
fixed polynomials of DESIGN.md §3.6 stand for.  The bar is north_star's own: >= 99.9 % of muons with equal flag and
step count, |dP|/P <= 1e-5 and |dr| <= 1e-5 m; two-sample KS p > 0.01 on final p, theta, x, y (on the whole
populations, and on the residual muons alone when there are at least 100 of them).
"""
import numpy as np
import pytest

from gpu_util import gpu_transport
from test_oracle_witness import check_against_witness

pytestmark = pytest.mark.gpu


def _witness(oracle, wl):
    return oracle.transport(oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom), wl.muons.pos_q, wl.muons.mom,
                            wl.seed, threads=oracle.max_threads(), libm=True)


def test_config1_full_against_libm_witness(mt, oracle, workloads):
    wl = workloads.config1(n_draws=200_000)                      # BASELINE configs[1]: 65 536 muons
    ref = _witness(oracle, wl)
    for sched in (2, 3):
        check_against_witness(gpu_transport(mt, wl, sched=sched), ref, "GPU config1 sched %d" % sched)


def test_config2_against_libm_witness(mt, oracle, workloads):
    # 30 m, ~720 steps per muon; 250k muons leave more than 100 residual muons, so the KS test on the residual subset
    # alone (north_star's rule for them) is exercised as well
    wl = workloads.config2(n=250_000, n_draws=100_000)
    c = check_against_witness(gpu_transport(mt, wl), _witness(oracle, wl), "GPU config2 (250k muons)")
    assert (~c["mask"]).sum() >= 100


def test_config3_small_against_libm_witness(mt, oracle, workloads):
    import torch
    wl = workloads.config3(n=100_000, n_draws=60_000, n_cells=2, half_width_cells=40, device="cuda")
    ref = _witness(oracle, wl)
    g = gpu_transport(mt, wl)                                    # default schedule: WAVEFRONT, lean kernel
    check_against_witness(g, ref, "GPU config3 small (100k muons, 80x80x750 grid)")
    del wl
    torch.cuda.empty_cache()


def test_joint_mode_against_libm_witness(mt, oracle, workloads):
    """The CUDA path with the paper's joint 2D tables held to the witness directly (VERDICT r2 next #3c): configs[1] in full
    under both persistent schedules, and the reduced field map under the default one (z-slab passes, joint LEAN kernel)."""
    import torch
    wl = workloads.config1(n_draws=200_000, joint=True)
    ref = _witness(oracle, wl)
    for sched in (2, 3):
        check_against_witness(gpu_transport(mt, wl, sched=sched), ref, "GPU config1 joint sched %d" % sched)
    wl = workloads.config3(n=100_000, n_draws=60_000, n_cells=2, half_width_cells=40, device="cuda", joint=True,
                           table_shape=(100, 64, 32))
    check_against_witness(gpu_transport(mt, wl), _witness(oracle, wl), "GPU config3 small joint (100k muons)")
    del wl
    torch.cuda.empty_cache()
