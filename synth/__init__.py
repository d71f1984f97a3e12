"""Seeded synthetic catalog generators shared by the oracle-side tests and the CUDA-side harness.

This package holds NONE of the method's arithmetic (no RA/Dec -> unit vector conversion, no
dot products, no binning, no estimator): it only emits sky positions as RA/Dec in degrees,
bin-edge *specifications* (nbins, min, max, mode) and seeded row subsets.  Both `oracle/`
and `paper_1204_6630_b200/` are fed from here; neither imports the other.
"""
from .catalogs import (  # noqa: F401
    CONFIGS,
    Config,
    SplitMix,
    make_config,
    subset_rows,
    uniform_patch,
    uniform_sphere,
    gaussian_clumps,
    neyman_scott,
    lognormal_mock,
    great_circle_ring,
    edges,
    config_edges,
    uniform_box,
    clustered_box,
    cubic_lattice,
    make_box_config,
)
