"""Seeded synthetic workloads shared by the CUDA path and the CPU oracle.

This package holds the INPUT GENERATORS only: shapes, seeds and value
distributions of the five BASELINE.json configs.  It contains none of the
method's arithmetic (no router GEMM, no gating, no counting, no objective):
both `paper_2606_15177_b200` (CUDA) and `oracle/` (CPU) consume the bytes
produced here and neither imports the other.

The paper measures on BurstGPT-derived traces with Qwen3-30B-A3B weights
(section 7.1); neither is available, so these generators stand
in for them with the shapes and skew the paper describes: heavy-tailed prompt
lengths (Fig. 1), few hot experts per layer (PAPER.md:67,
Fig. 3) and source-dependent expert skew (Fig. 4).  The recipe is
stated in DESIGN.md section 4.
"""
from .configs import RouterCfg, Workload, WORKLOADS, get_workload, scaled  # noqa: F401
from . import gen  # noqa: F401
