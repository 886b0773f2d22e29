"""B200-native muon transport by histogram sampling (arxiv 2512.10520): the per-muon step loop as
hand-written CUDA behind a C ABI (include/muon_transport.h).

    from paper_2512_10520_b200 import binding, workloads, build

`binding` loads libmuon_transport.so lazily and raises if it is missing; nothing here falls back to a CPU path.
"""
from . import workloads  # noqa: F401  (numpy only)
from . import build      # noqa: F401
from . import binding    # noqa: F401  (loads the shared library on first use)
