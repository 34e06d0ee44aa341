"""The five workloads of BASELINE.json `configs`, as parameters.

PAPER.md:101 (§4): "50 alternating box-shaped layers of absorber and gap
material"; materials, thicknesses, energies, seeds and buffer sizes are
BASELINE.json's.  DESIGN.md §"Input recipe" states how these stand in for the
paper's AdePT example19 / TestEm3 runs.
"""
from __future__ import annotations

from dataclasses import dataclass

from .tables import TableSet, build_tables


@dataclass(frozen=True)
class Geometry:
    n_layers: int
    abs_mm: float = 2.3         # Pb absorber
    gap_mm: float = 5.7         # liquid-Ar gap
    half_xy_mm: float = 200.0
    mat_abs: int = 0
    mat_gap: int = 1


E_CUT = 0.1     # MeV, production = tracking cut (all configs)

CONFIGS = {
    # name: parameters.  kind: 0 = e-, 1 = e+, 2 = gamma
    "tiny": dict(seed=1, n_layers=4, half_xy_mm=50.0, n_bins=64, e_max=100.0,
                 n_primaries=16, e_primary=10.0, scheme="dense", capacity=4096),
    "full": dict(seed=2, n_layers=50, half_xy_mm=200.0, n_bins=256, e_max=1.0e4,
                 n_primaries=1000, e_primary=1000.0, scheme="dense", capacity=2 * 1024 * 1024),
    "single_step": dict(seed=3, n_layers=50, half_xy_mm=200.0, n_bins=256, e_max=1.0e4,
                        n_tracks=1 << 24, fractions=(0.4, 0.1, 0.5)),
    "sweep": dict(seed=4, n_layers=50, half_xy_mm=200.0, n_bins=256, e_max=1.0e4,
                  span=4 * 1024 * 1024, reserve=512 * 1024,
                  occupancies=(0.1, 0.3, 0.5, 0.7, 0.9), spawn_fraction=0.05),
    "heavy": dict(seed=5, n_layers=50, half_xy_mm=200.0, n_bins=256, e_max=1.0e4,
                  n_primaries=10000, e_primary=1.0e4, scheme="dense", capacity=8 * 1024 * 1024),
}


def geometry_for(name: str) -> Geometry:
    c = CONFIGS[name]
    return Geometry(n_layers=c["n_layers"], half_xy_mm=c["half_xy_mm"])


_TABLE_CACHE: dict = {}


def tables_for(name: str, physics: int = 0) -> TableSet:
    """Tables of a config; physics = 1: the extended rule set (DESIGN.md rules X35-X39)."""
    c = CONFIGS[name]
    key = (c["n_bins"], c["e_max"], physics)
    if key not in _TABLE_CACHE:
        _TABLE_CACHE[key] = build_tables(c["n_bins"], E_CUT, c["e_max"], E_CUT, physics=physics)
    return _TABLE_CACHE[key]
