"""CPU-side checks of the boundary: the C-ABI library builds, loads, and exports every symbol the header
declares; the binding's structs have the header's layout; without a GPU the product path fails loudly."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "muon_transport.h")
PROBES_HEADER = os.path.join(ROOT, "include", "muon_probes.h")


def declared_functions(header=HEADER):
    src = open(header).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mt_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(mt):
    names = declared_functions()
    assert {"mt_load_histograms", "mt_build_alias", "mt_set_geometry", "mt_transport"} <= set(names)
    L = ctypes.CDLL(mt.binding.LIB_PATH)
    for n in names:
        assert hasattr(L, n), n
    assert sorted(mt.binding.SYMBOLS) == names


def test_probes_live_in_their_own_library(mt):
    """include/ holds two headers and each has its library: the measurement probes (include/muon_probes.h) are exported by
    libmuon_probes.so and by it alone — the product boundary carries the transport calls and their documented hooks only."""
    assert sorted(f for f in os.listdir(os.path.join(ROOT, "include")) if f.endswith(".h")) == ["muon_probes.h", "muon_transport.h"]
    names = declared_functions(PROBES_HEADER)
    assert names == sorted(mt.binding.PROBE_SYMBOLS) == ["mt_measure_peaks", "mt_probe_field_paths"]
    P = ctypes.CDLL(mt.binding.PROBES_LIB_PATH)
    L = ctypes.CDLL(mt.binding.LIB_PATH)
    for n in names:
        assert hasattr(P, n), n
        assert not hasattr(L, n), n
    for n in declared_functions():                       # and nothing of the transport ABI leaks into the probes' library
        assert not hasattr(P, n), n


def test_struct_layouts_match_the_header(mt):
    b = mt.binding
    assert ctypes.sizeof(b.mt_region) == 40
    assert ctypes.sizeof(b.mt_hist_desc) == 24 + 5 * 8 + 8 and b.mt_hist_desc.hist_mode.offset == 64
    assert b.mt_geometry.regions.offset == 48 and b.mt_geometry.d_material.offset == 88
    assert ctypes.sizeof(b.mt_geometry) == 128 and b.mt_geometry.field_mode.offset == 104 and b.mt_geometry.exit_mode.offset == 120
    assert b.mt_geometry.n_blocks.offset == 108 and b.mt_geometry.blocks.offset == 112
    assert ctypes.sizeof(b.mt_poly_block) == 88 and b.mt_poly_block.xy_hi.offset == 40 and b.mt_poly_block.material.offset == 72
    from paper_2512_10520_b200.workloads import POLY_DTYPE, REGION_DTYPE
    assert POLY_DTYPE.itemsize == 88 and POLY_DTYPE.fields["xy_hi"][1] == 40 and REGION_DTYPE.itemsize == 40
    assert ctypes.sizeof(b.mt_muons_in) == 16 and ctypes.sizeof(b.mt_muons_out) == 48
    assert b.lib().mt_strerror(b.MT_ERR_EMPTY_HIST).decode().startswith("empty")


def test_no_cpu_fallback(mt):
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU box")
    with pytest.raises(mt.binding.MtError):
        mt.binding.mt_create(0)
    with pytest.raises(RuntimeError):
        mt.binding.MuonTransport(0)


def test_product_path_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2512_10520_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "muon_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2512_10520_b200", text, flags=re.M), f
            assert "csrc/" not in text.replace("paper_2512_10520_b200/csrc/.", "") or f.endswith(".cpp")
