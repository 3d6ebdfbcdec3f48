"""ORACLE package: test infrastructure, not product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this.  It never imports paper_2409_04668_b200 and shares no code with it.
"""
from .lattice import expand_lattice, translate_quadric  # noqa: F401
from .binding import Oracle, build, lib_path, philox4x32_10, draws, source_key, child_key, mix64, surface_distance  # noqa: F401
