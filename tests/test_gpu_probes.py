"""-m gpu: the in-process probes behind bench.py's roofline.measured_peaks (include/muon_probes.h, libmuon_probes.so:
csrc/mt_probe.cu, mt_probe_field.cu — a library of their own, not part of the transport boundary) return
numbers that are physically ordered and inside the hardware's envelope — a probe whose loop the compiler deleted, or one
that timed an empty launch, shows up here as a rate above what 148 SMs can issue."""
import pytest

pytestmark = pytest.mark.gpu


def test_measured_peaks_are_ordered_and_bounded(mt):
    b = mt.binding
    p = b.mt_measure_peaks(0)
    nominal = p["sm_count"] * 128 * p["sm_clock_mhz_nominal"] * 1e6           # one thread-op per lane per clock
    ffma = p["ffma_thread_ops_per_s"]
    assert 0.40 * nominal < ffma <= 1.001 * nominal                          # (a power-capped box clocks lower, never higher)
    # relative to the FP32 stream of the same moment: the 16-lane pipes run at half its rate, the wide multiply and the
    # special-function unit below that
    assert 0.40 < p["lop3_thread_ops_per_s"] / ffma < 0.65
    assert 0.40 < p["imad_thread_ops_per_s"] / ffma < 0.65
    assert 0.10 < p["mulhi_thread_ops_per_s"] / ffma < 0.45
    assert 0.05 < p["mufu_thread_ops_per_s"] / ffma < 0.35
    # mixed streams: the ALU pipe runs beside the FP32 stream (12 instructions in about the time of the 8
    # fma alone would be 1.5x; anything above 0.85 of the fma rate shows the overlap), the FMA pipe's integer half does not:
    # 8 fma + 4 mad.lo cost 8 + 4 x 2 cycles (0.75), 8 fma + 2 mul.wide 8 + 2 x 4 (0.625)
    assert 0.85 < p["mix_ffma8_lop3_4_thread_ops_per_s"] / ffma < 1.05
    assert 0.60 < p["mix_ffma8_imad4_thread_ops_per_s"] / ffma < 0.85
    assert 0.45 < p["mix_ffma8_mulwide2_thread_ops_per_s"] / ffma < 0.75
    # gathers: L1-resident > L2-resident > HBM, the last below the pool's measured copy bandwidth
    assert p["gather_l1_bytes_per_s"] > p["gather_64m_bytes_per_s"] > p["gather_1400m_bytes_per_s"] > 2e11
    assert abs(p["gather_675k_bytes_per_s"] / p["gather_64m_bytes_per_s"] - 1.0) < 0.25     # both L2-resident
    assert p["gather_1400m_bytes_per_s"] < 8e12 and p["gather_l1_bytes_per_s"] < 148 * 128 * 2.1e9


def test_field_path_probe(mt):
    b = mt.binding
    f = b.mt_probe_field_paths(0)
    assert f["records_per_launch"] == 148 * 3 * 16 * 256 * 64 * 4 or f["records_per_launch"] > 1e8
    assert f["ldg_records_per_s"] > 0 and f["tex_records_per_s"] > 0 and f["tma_records_per_s"] > 0
    # what DESIGN.md §7 concludes from it: plain read-only loads are the fastest of the three on the step loop's pattern
    assert f["ldg_records_per_s"] > f["tma_records_per_s"] > 0.5 * f["tex_records_per_s"]
    assert f["ldg_records_per_s"] * 32 < 148 * 128 * 2.1e9 * 2                    # below the L1 data path's envelope
