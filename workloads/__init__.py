"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds *input data generators only*: the analytic cross-section
tables (BASELINE.json configs: "built from analytic forms"), the slab
calorimeter description (§4) and the seeded track populations
of BASELINE.json configs 3 and 4.  It contains none of the transport
arithmetic (no Philox, no lg/ex, no step logic) and imports neither
``oracle`` nor ``paper_2302_08252_b200``.
"""
from .configs import CONFIGS, Geometry, geometry_for, tables_for  # noqa: F401
from .tables import MATERIALS, TableSet, build_tables  # noqa: F401
from .tracks import TRACK_DTYPE, PRIMARY_DTYPE, gen_tracks, gen_primaries, gen_sweep  # noqa: F401
