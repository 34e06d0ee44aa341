"""Seeded synthetic track populations (BASELINE.json configs 3 and 4) and
primary guns (configs 1, 2, 5).

Pure input data: numpy's PCG64 stream `default_rng(seed)`, float64 maths,
one rounding to float32.  Track ids are unique 64-bit labels made from the
track index by an odd-multiplier bijection (they are inputs: the method only
requires them to be distinct).  Nothing here belongs to the transport step.
"""
from __future__ import annotations

import math

import numpy as np

from .configs import CONFIGS, E_CUT, Geometry, geometry_for

# 56-byte record, identical to `adept_track` in include/adept.h
TRACK_DTYPE = np.dtype([
    ("pos", "<f4", (3,)), ("dir", "<f4", (3,)), ("ekin", "<f4"), ("nial", "<f4", (3,)),
    ("vol", "<u4"), ("id_lo", "<u4"), ("id_hi", "<u4"), ("step", "<u4")], align=False)
assert TRACK_DTYPE.itemsize == 56

# 32-byte record, identical to `adept_primary`
PRIMARY_DTYPE = np.dtype([
    ("kind", "<u4"), ("pos", "<f4", (3,)), ("dir", "<f4", (3,)), ("ekin", "<f4")], align=False)
assert PRIMARY_DTYPE.itemsize == 32

_ID_MUL = np.uint64(0x9E3779B97F4A7C15)
_SEED_MUL = np.uint64(0xD1B54A32D192ED03)


def _ids(first_index: int, n: int, seed: int):
    with np.errstate(over="ignore"):
        i = np.arange(first_index + 1, first_index + 1 + n, dtype=np.uint64)
        v = i * _ID_MUL + np.uint64(seed) * _SEED_MUL
    return (v & np.uint64(0xFFFFFFFF)).astype(np.uint32), (v >> np.uint64(32)).astype(np.uint32)


def _fill_phase_space(rng: np.random.Generator, out: np.ndarray, geo: Geometry, e_max: float):
    """Positions uniform in the calorimeter, isotropic directions, log-uniform
    kinetic energies, exponential(1) interaction lengths (config 3)."""
    n = out.shape[0]
    a, g = np.float32(geo.abs_mm), np.float32(geo.gap_mm)
    pitch = float(np.float32(a + g))
    depth = geo.n_layers * pitch
    z = (rng.random(n) * depth).astype(np.float32)
    x = ((2.0 * rng.random(n) - 1.0) * geo.half_xy_mm).astype(np.float32)
    y = ((2.0 * rng.random(n) - 1.0) * geo.half_xy_mm).astype(np.float32)
    out["pos"][:, 0], out["pos"][:, 1], out["pos"][:, 2] = x, y, z
    z64 = z.astype(np.float64)
    layer = np.minimum((z64 / pitch).astype(np.int64), geo.n_layers - 1)
    in_gap = (z64 - layer * pitch) >= float(a)
    out["vol"] = (2 * layer + in_gap).astype(np.uint32)
    ct = 1.0 - 2.0 * rng.random(n)
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    phi = 2.0 * math.pi * rng.random(n)
    out["dir"][:, 0] = (st * np.cos(phi)).astype(np.float32)
    out["dir"][:, 1] = (st * np.sin(phi)).astype(np.float32)
    out["dir"][:, 2] = ct.astype(np.float32)
    e = E_CUT * np.exp(rng.random(n) * math.log(e_max / E_CUT))
    out["ekin"] = np.clip(e, E_CUT, e_max).astype(np.float32)
    out["ekin"] = np.clip(out["ekin"], np.float32(E_CUT), np.float32(e_max))
    u = 1.0 - rng.random((n, 3))          # (0, 1]
    out["nial"] = np.maximum(-np.log(u), 1e-30).astype(np.float32)
    out["step"] = 0


def gen_tracks(n_total: int, seed: int, geo: Geometry, e_max: float,
               fractions=(0.4, 0.1, 0.5)):
    """Config 3: returns [tracks_e-, tracks_e+, tracks_gamma] (TRACK_DTYPE)."""
    n0 = int(round(n_total * fractions[0]))
    n1 = int(round(n_total * fractions[1]))
    counts = (n0, n1, n_total - n0 - n1)
    rng = np.random.default_rng(seed)
    out, first = [], 0
    for k, nk in enumerate(counts):
        t = np.zeros(nk, dtype=TRACK_DTYPE)
        _fill_phase_space(rng, t, geo, e_max)
        t["id_lo"], t["id_hi"] = _ids(first, nk, seed)
        first += nk
        out.append(t)
    return out


def gen_single_step(n_total: int | None = None):
    c = CONFIGS["single_step"]
    return gen_tracks(n_total or c["n_tracks"], c["seed"], geometry_for("single_step"),
                      c["e_max"], c["fractions"])


def gen_sweep(occupancy: float, *, span: int | None = None, seed: int | None = None,
              spawn_fraction: float | None = None, shuffled: bool = False):
    """Config 4: per kind, `round(occupancy*span)` live tracks.

    Returns a list of 3 dicts {tracks, slots, forced}: `slots` is an ascending
    uniformly random subset of [0, span) (the sparse single buffer's live
    slots; the dense double buffer ignores it and packs), `forced` marks the
    tracks that must spawn exactly one secondary this step (nial of brems /
    photoelectric = 1e-30); all other used nial are 1e6 (no interaction).
    """
    c = CONFIGS["sweep"]
    span = span or c["span"]
    seed = c["seed"] if seed is None else seed
    spawn_fraction = c["spawn_fraction"] if spawn_fraction is None else spawn_fraction
    geo = geometry_for("sweep")
    rng = np.random.default_rng([seed, int(round(occupancy * 1000))])
    n_live = int(round(occupancy * span))
    out, first = [], 0
    for kind in range(3):
        t = np.zeros(n_live, dtype=TRACK_DTYPE)
        _fill_phase_space(rng, t, geo, c["e_max"])
        forced = rng.random(n_live) < spawn_fraction
        if kind < 2:
            # brems needs Sigma_brems > 0: re-draw forced e+- sitting on the cut
            low = forced & (t["ekin"] <= np.float32(E_CUT * (1.0 + 1e-3)))
            while low.any():
                e = E_CUT * np.exp(rng.random(int(low.sum())) * math.log(c["e_max"] / E_CUT))
                t["ekin"][low] = np.clip(e, E_CUT, c["e_max"]).astype(np.float32)
                low = forced & (t["ekin"] <= np.float32(E_CUT * (1.0 + 1e-3)))
        t["nial"] = np.float32(1e6)
        jstar = 0 if kind < 2 else 2
        t["nial"][forced, jstar] = np.float32(1e-30)
        t["id_lo"], t["id_hi"] = _ids(first, n_live, seed + 1000 * int(round(occupancy * 100)))
        first += n_live
        slots = np.sort(rng.choice(span, size=n_live, replace=False)).astype(np.uint32)
        if shuffled:
            rng.shuffle(slots)
        out.append(dict(tracks=t, slots=slots, forced=forced))
    return out


def gen_primaries(n: int, e_primary: float, kind: int = 0):
    """Particle gun of configs 1, 2, 5: normal incidence at the origin."""
    p = np.zeros(n, dtype=PRIMARY_DTYPE)
    p["kind"] = kind
    p["dir"][:, 2] = 1.0
    p["ekin"] = np.float32(e_primary)
    return p
