"""Seeded synthetic input generators for the five BASELINE.json workloads.

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_02455_b200/``).  It holds geometry, topology, parameter tables and
random weights only -- none of the method's arithmetic (no force field, no
integrator, no Philox, no transport map).  See DESIGN.md "Input recipe".
"""
from .workloads import (  # noqa: F401
    Workload, Potential, Mlip, make_workload, WORKLOADS, mlip_weight_count,
    mlip_weight_offsets, K_B, AMU, to_soa, from_soa, with_target_as_draft,
    tile_periodic, make_mlip, PAIR_COLS,
)
