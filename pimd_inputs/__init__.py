"""Seeded synthetic inputs for the PIMD hot path.

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2503_23728_b200/`).  It holds no arithmetic of the method itself
(no neighbour search, no network evaluation, no integrator): it only builds
geometries, the packed random-init weight blob and the scalar run parameters
of the five workloads named in BASELINE.json `configs`.

The inputs stand in for the paper's formic-acid-dimer and water/ice systems
(PAPER.md L158-L253), whose datasets and trained weights are not available;
nothing here is taken from those datasets.
"""
from .workloads import (  # noqa: F401
    Workload,
    NetSpec,
    MASSES_AMU,
    SPECIES_H,
    SPECIES_C,
    SPECIES_O,
    make_workload,
    workload_names,
    pack_weights,
    n_weights,
    weight_layout,
    fad_geometry,
    water_geometry,
    ice_ic_geometry,
)
