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


def philox4x32_10_np(ctr, key):
    """Philox-4x32-10 (Salmon et al., SC'11) written out in numpy from the published description
    (DESIGN.md rule R1) -- independent of the oracle's and the library's routines, and pinned to
    the same known-answer vectors (tests/golden/philox4x32_10_kat.txt) by test_oracle_rng_math.py.
    ctr [n][4], key [n][2] uint32 -> [n][4] uint32."""
    c = np.array(ctr, dtype=np.uint64).reshape(-1, 4).copy()
    k = np.array(key, dtype=np.uint64).reshape(-1, 2).copy()
    m0, m1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
    w0, w1 = np.uint64(0x9E3779B9), np.uint64(0xBB67AE85)
    mask, sh = np.uint64(0xFFFFFFFF), np.uint64(32)
    for _ in range(10):
        p0 = m0 * c[:, 0]
        p1 = m1 * c[:, 2]
        n0 = (p1 >> sh) ^ c[:, 1] ^ k[:, 0]
        n1 = p1 & mask
        n2 = (p0 >> sh) ^ c[:, 3] ^ k[:, 1]
        n3 = p0 & mask
        c = np.stack([n0, n1, n2, n3], 1)
        k[:, 0] = (k[:, 0] + w0) & mask
        k[:, 1] = (k[:, 1] + w1) & mask
    return c.astype(np.uint32)


def primary_ids_np(indices, seed):
    """Rule R4 as DESIGN.md words it: (id_lo, id_hi) = words 0, 1 of
    Philox(counter = (p_lo, p_hi, 0, 0x5052494D), key = (seed_lo, seed_hi))."""
    p = np.asarray(indices, dtype=np.uint64)
    ctr = np.zeros((p.shape[0], 4), dtype=np.uint64)
    ctr[:, 0] = p & np.uint64(0xFFFFFFFF)
    ctr[:, 1] = p >> np.uint64(32)
    ctr[:, 3] = 0x5052494D
    key = np.zeros((p.shape[0], 2), dtype=np.uint64)
    key[:, 0] = np.uint64(seed) & np.uint64(0xFFFFFFFF)
    key[:, 1] = np.uint64(seed) >> np.uint64(32)
    w = philox4x32_10_np(ctr, key)
    return w[:, 0], w[:, 1]
