"""Seeded synthetic workload generators (BASELINE.json configs 1-5).

TEST / BENCH INFRASTRUCTURE shared by the oracle harness and the CUDA harness.  This package
holds none of the method's arithmetic: it only produces inputs (CSR matrices, bounds, boxes,
phantoms).  Everything is generated in fp64 and rounded ONCE to fp32; those fp32 arrays are
*the* input of both sides (the oracle widens them exactly to fp64).

Recipes: DESIGN.md section "Input recipe"; SURVEY.md section 8(d).
"""
from .workloads import (  # noqa: F401
    Problem,
    build_native,
    ct_matrix,
    segment_matrix,
    imrt_matrix,
    random_csr,
    config1_tiny_ct,
    config2_crosswell,
    config3_lowdose_ct,
    config4_imrt,
    config5_sweep_point,
    interleaved_angle_blocks,
    SEED0,
)
