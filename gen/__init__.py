"""Seeded synthetic input generators (BASELINE.json:configs).

This package serves BOTH the fp64 oracle (`oracle/`) and the CUDA path
(`paper_2310_03121_b200/`).  It holds none of the method's arithmetic: it only
draws positions / species / upstream gradients / weights with the shapes and
statistics of the paper's workloads (PAPER.md:183-185 ligand ML region,
PAPER.md:164 DHFR-sized solvated box) and rejects geometries that sit within
1e-4 A of a cutoff (BASELINE.json:north_star).
"""
from .workloads import (  # noqa: F401
    AniParams,
    ani1x_style_params,
    ani2x_shaped_params,
    make_c1,
    make_c2,
    make_water_box,
    make_periodic_cell,
    make_c3,
    make_c4,
    make_c5_weights,
    make_ensemble_weights,
    make_workload,
    random_walk,
    Workload,
)
