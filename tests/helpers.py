"""Helpers shared by the test modules (no transport arithmetic of their own)."""
import numpy as np

from workloads import TRACK_DTYPE


def make_tracks(n, *, pos=(0.0, 0.0, 0.0), dir=(0.0, 0.0, 1.0), ekin=1.0, nial=(-1.0, -1.0, -1.0),
                vol=0, id0=1, step=0):
    t = np.zeros(n, dtype=TRACK_DTYPE)
    t["pos"] = np.asarray(pos, dtype=np.float32)
    t["dir"] = np.asarray(dir, dtype=np.float32)
    t["ekin"] = np.float32(ekin) if np.isscalar(ekin) else np.asarray(ekin, dtype=np.float32)
    t["nial"] = np.asarray(nial, dtype=np.float32)
    t["vol"] = vol
    ids = np.arange(id0, id0 + n, dtype=np.uint64) * np.uint64(0x9E3779B97F4A7C15)
    t["id_lo"] = (ids & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    t["id_hi"] = (ids >> np.uint64(32)).astype(np.uint32)
    t["step"] = step
    return t


def sort_by_id(t):
    key = t["id_hi"].astype(np.uint64) << np.uint64(32) | t["id_lo"].astype(np.uint64)
    return t[np.argsort(key, kind="stable")]


def ulp_diff(a32, ref64):
    """|a - ref| in units of ulp(ref) for float32 `a32` vs float64 reference."""
    a32 = np.asarray(a32, dtype=np.float32)
    ref32 = np.asarray(ref64, dtype=np.float64).astype(np.float32)
    ulp = np.spacing(np.abs(ref32)).astype(np.float64)
    return np.abs(a32.astype(np.float64) - np.asarray(ref64, dtype=np.float64)) / ulp
