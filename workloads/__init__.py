"""Seeded synthetic problem descriptions (SURVEY.md Appendix C / BASELINE.json configs).

This module holds *inputs only*: geometry tables, cross sections, source, mesh and
time grids as plain numpy arrays.  It contains none of the transport arithmetic and is
the single piece of Python both the oracle binding (oracle/) and the CUDA binding
(paper_2409_04668_b200/) consume.  Neither of those imports the other.
"""
from .configs import (  # noqa: F401
    Problem,
    config0_infinite_medium,
    config1_slab,
    config1a_pure_absorber_beam,
    config2_lduct,
    config3_pin_lattice,
    config3_xs,
    infinite_medium_multigroup,
    run_seed,
    CONFIGS,
    get_config,
)
