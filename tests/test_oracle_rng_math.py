"""Pins for the oracle's random numbers and elementary functions
(DESIGN.md rules R1, R3, M8, M9, M10, S27).  CPU only.

Philox is pinned to the published known-answer vectors; the fp32 elementary
functions are pinned to the mathematical functions evaluated in float64 by
numpy/libm (an independent implementation), with the error bounds DESIGN.md
states.
"""
import math
import os

import numpy as np
import pytest

from oracle import math_fns
from tests.helpers import philox4x32_10_np, ulp_diff

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answer_vectors():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = math_fns.philox(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_numpy_philox_of_the_test_helpers_passes_the_same_vectors():
    """tests/helpers.py philox4x32_10_np (used to pin rule R4 independently of the oracle's routine)
    against the published vectors, and the oracle against it on random inputs."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    for r in rows:
        v = [int(x, 16) for x in r]
        assert [int(x) for x in philox4x32_10_np([v[0:4]], [v[4:6]])[0]] == v[6:10]
    rng = np.random.default_rng(1)
    ctr = rng.integers(0, 2**32, size=(5000, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(5000, 2), dtype=np.uint64).astype(np.uint32)
    assert (math_fns.philox_array(ctr, key) == philox4x32_10_np(ctr, key)).all()


def test_philox_array_matches_scalar_and_is_a_bijection_sample():
    rng = np.random.default_rng(0)
    ctr = rng.integers(0, 2**32, size=(1000, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(1000, 2), dtype=np.uint64).astype(np.uint32)
    out = math_fns.philox_array(ctr, key)
    for i in (0, 17, 999):
        assert (out[i] == math_fns.philox(ctr[i], key[i])).all()
    # a counter-mode bijection: distinct counters under one key give distinct blocks
    ctr2 = np.zeros((4096, 4), dtype=np.uint32)
    ctr2[:, 0] = np.arange(4096)
    key2 = np.tile(np.array([[123, 456]], dtype=np.uint32), (4096, 1))
    blocks = math_fns.philox_array(ctr2, key2)
    assert len({tuple(b) for b in blocks}) == 4096
    # crude uniformity: mean of the top bit over 16384 words within 5 sigma
    bits = (blocks >> 31).astype(np.float64)
    assert abs(bits.mean() - 0.5) < 5 * 0.5 / math.sqrt(bits.size)


def test_u01_grid_exhaustive():
    # R3: every one of the 2^23 outputs is an odd multiple of 2^-24 in (0,1), all distinct
    x = (np.arange(1 << 23, dtype=np.uint64) << np.uint64(9)).astype(np.uint32)
    u = math_fns.u01(x)
    k = u.astype(np.float64) * 2.0**24
    assert (k == np.floor(k)).all()
    assert (k.astype(np.int64) == 2 * np.arange(1 << 23, dtype=np.int64) + 1).all()
    assert u.min() == np.float32(2.0**-24) and u.max() == np.float32(1 - 2.0**-24)
    # low 9 bits are ignored
    assert (math_fns.u01(x[:1000] | np.uint32(0x1FF)) == u[:1000]).all()


def _float_sweep(lo, hi, stride):
    a = np.float32(lo).view(np.uint32)
    b = np.float32(hi).view(np.uint32)
    return np.arange(int(a), int(b), stride, dtype=np.uint32).view(np.float32)


def _every_float(lo, hi, chunk=1 << 23):
    """Every fp32 in [lo, hi), in chunks (exhaustive sweep of the used domain)."""
    a, b = int(np.float32(lo).view(np.uint32)), int(np.float32(hi).view(np.uint32))
    for first in range(a, b, chunk):
        yield np.arange(first, min(first + chunk, b), dtype=np.uint32).view(np.float32)


def test_lg_against_libm():
    # M8: <= 2 ulp on EVERY fp32 of the used domain [1e-8, 1e5]; the u grid gives finite positive -lg(u)
    n = 0
    for x in _every_float(1e-8, 1e5):
        y = math_fns.lg(x)
        ref = np.log(x.astype(np.float64))
        nz = ref != 0
        # absolute floor of 2^-24 near x = 1 (ln is ~1e-7 there and the result comes from s = (m-1)/(m+1))
        err = np.abs(y[nz].astype(np.float64) - ref[nz])
        ok = (ulp_diff(y[nz], ref[nz]) <= 2.0) | (err <= 2.0**-24 * 0.5)
        assert ok.all(), (x[nz][~ok][:5], y[nz][~ok][:5])
        n += x.shape[0]
    assert n > 3.6e8
    assert math_fns.lg(np.float32([1.0]))[0] == 0.0
    # exhaustive over the u grid: finite, positive, monotone non-increasing in u
    xs = (np.arange(1 << 23, dtype=np.uint64) << np.uint64(9)).astype(np.uint32)
    e = -math_fns.lg(math_fns.u01(xs))
    assert np.isfinite(e).all() and (e > 0).all()
    assert e.max() < 16.7 and e.min() > 5.9e-8
    assert (np.diff(e) <= 0).all()


def test_ex_against_libm():
    # M9: <= 1 ulp on EVERY fp32 of [-20, -1e-6] and [1e-6, 12] (the step uses [-17, 11.6]), and 0
    n = 0
    for sign, hi in ((1.0, 12.0), (-1.0, 20.0)):
        for x in _every_float(1e-6, hi):
            x = np.float32(sign) * x
            assert ulp_diff(math_fns.ex(x), np.exp(x.astype(np.float64))).max() <= 1.0
            n += x.shape[0]
    assert n > 3.9e8
    assert math_fns.ex(np.float32([0.0]))[0] == 1.0


def test_sincos2pi_against_libm():
    # M10: abs error <= 1e-7, |sin^2 + cos^2 - 1| <= 2e-7; exact at quadrant points
    xs = (np.arange(0, 1 << 23, 1, dtype=np.uint64) << np.uint64(9)).astype(np.uint32)   # the whole u grid
    u = math_fns.u01(xs)
    s, c = math_fns.sincos2pi(u)
    a = 2.0 * math.pi * u.astype(np.float64)
    assert np.abs(s - np.sin(a)).max() <= 1.0e-7
    assert np.abs(c - np.cos(a)).max() <= 1.0e-7
    assert np.abs(s.astype(np.float64) ** 2 + c.astype(np.float64) ** 2 - 1).max() <= 2e-7
    s, c = math_fns.sincos2pi(np.float32([0.25, 0.5, 0.75]))
    assert list(s) == [1.0, 0.0, -1.0] or np.allclose(s, [1, 0, -1], atol=0)
    assert np.allclose(c, [0, -1, 0], atol=0)


def test_rotate_is_a_rotation():
    # S27: |d'| = 1, d.d' = cos(theta); azimuth changes the component normal to d
    rng = np.random.default_rng(5)
    n = 20000
    ct0 = rng.uniform(-1, 1, n)
    ph0 = rng.uniform(0, 2 * math.pi, n)
    d = np.stack([np.sqrt(1 - ct0**2) * np.cos(ph0), np.sqrt(1 - ct0**2) * np.sin(ph0), ct0], 1)
    d[:10] = [0, 0, 1]
    d[10:20] = [0, 0, -1]
    d = d.astype(np.float32)
    d /= np.linalg.norm(d.astype(np.float64), axis=1, keepdims=True).astype(np.float32)
    ct = rng.uniform(-1, 1, n).astype(np.float32)
    st = np.sqrt(1 - ct.astype(np.float64) ** 2).astype(np.float32)
    phi = rng.uniform(0, 2 * math.pi, n)
    out = math_fns.rotate(d, st, ct, np.sin(phi).astype(np.float32), np.cos(phi).astype(np.float32))
    o64, d64 = out.astype(np.float64), d.astype(np.float64)
    assert np.abs(np.linalg.norm(o64, axis=1) - 1).max() < 3e-7
    # away from the poles of d the polar angle is reproduced to rounding; within 1e-3 of a pole
    # sp = sqrt(1 - dz^2) inherits the fp32 normalisation error of d (relative error ~1e-7 / sp^2)
    dot_err = np.abs((o64 * d64).sum(1) - ct)
    sp2 = np.maximum(1.0 - d64[:, 2] ** 2, 1e-10)
    far = sp2 > 0.02
    assert (dot_err < 2e-6 + 4e-7 / sp2).all()
    assert dot_err[far].max() < 2.5e-5
    # phi and phi + pi give mirror images about d:  d'(phi) + d'(phi+pi) = 2 cos(theta) d
    out2 = math_fns.rotate(d, st, ct, -np.sin(phi).astype(np.float32), -np.cos(phi).astype(np.float32))
    assert np.abs(o64 + out2.astype(np.float64) - 2 * ct[:, None] * d64)[far].max() < 5e-5
    # explicit value: d = x, theta = 90 deg, phi = 0  ->  u = (dx dz c - dy s, ..., -sp c) = (0, 0, -1)
    o = math_fns.rotate(np.float32([[1, 0, 0]]), 1.0, 0.0, 0.0, 1.0)
    assert np.allclose(o, [[0, 0, -1]], atol=1e-7)
    # d = z: d' = (st cphi, st sphi, ct)
    o = math_fns.rotate(np.float32([[0, 0, 1]]), 0.6, 0.8, 1.0, 0.0)
    assert np.allclose(o, [[0, 0.6, 0.8]], atol=1e-7)
