"""fp64 CPU oracle of the PrefixFlow attention hot path.  TEST INFRASTRUCTURE, not product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2606_01143_b200 except seeded input shapes
handed to it by the caller, and the CUDA path never imports it.
"""
from .reference import (  # noqa: F401
    build, lib, max_threads, widen, fullseq, rows, cols, group_reference, GroupReference,
    sampled_phaseB, sampled_rows,
)
from .companions import rope, kv_proj_grad  # noqa: F401
