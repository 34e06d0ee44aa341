"""ctypes access to oracle/adept_oracle.cpp (built with g++, no CUDA).

ORACLE — test infrastructure.  Compile flags are part of the arithmetic
contract (DESIGN.md rule M7): -O2 -ffp-contract=off, no -ffast-math, plain
x86-64 so the same .so runs on any host.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "adept_oracle.cpp")
_SO = os.path.join(_HERE, "libadept_oracle.so")
_LOCK = threading.Lock()
_LIB = None

CXXFLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
            "-Wall", "-Wextra"]

TRACE_DTYPE = np.dtype([("id_lo", "<u4"), ("id_hi", "<u4"), ("step", "<u4"), ("kind", "<u4"),
                        ("winner", "<i4"), ("margin", "<f4")])


class _Geometry(C.Structure):
    _fields_ = [("n_layers", C.c_uint32), ("abs_mm", C.c_float), ("gap_mm", C.c_float),
                ("half_xy_mm", C.c_float), ("mat_abs", C.c_uint32), ("mat_gap", C.c_uint32)]


class _Tables(C.Structure):
    _fields_ = [("n_bins", C.c_uint32), ("n_materials", C.c_uint32), ("e_min", C.c_float),
                ("e_max", C.c_float), ("ln_e_min", C.c_float), ("inv_dln", C.c_float),
                ("e_cut", C.c_float), ("data", C.POINTER(C.c_float)),
                ("physics", C.c_uint32), ("data_x", C.POINTER(C.c_float))]


class _Result(C.Structure):
    _fields_ = [("live", C.c_uint64 * 3), ("steps", C.c_uint64 * 3), ("secondaries", C.c_uint64 * 3),
                ("killed", C.c_uint64 * 3), ("escaped_n", C.c_uint64 * 3),
                ("slots_used", C.c_uint64 * 3), ("iterations", C.c_uint64),
                ("e_injected", C.c_double), ("e_escaped", C.c_double),
                ("e_escaped_kind", C.c_double * 3)]


def build(force: bool = False) -> str:
    """Compile the oracle with g++ if the .so is missing or stale."""
    with _LOCK:
        stale = (not os.path.exists(_SO)) or os.path.getmtime(_SO) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _SO + ".tmp%d" % os.getpid()
            subprocess.run(["g++", *CXXFLAGS, "-o", tmp, _SRC], check=True)
            os.replace(tmp, _SO)
    return _SO


def lib():
    global _LIB
    if _LIB is None:
        L = C.CDLL(build())
        vp, u64, u32 = C.c_void_p, C.c_uint64, C.c_uint32
        L.orc_create.restype = vp
        L.orc_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Tables), u64]
        L.orc_destroy.argtypes = [vp]
        for name in ("orc_inject", "orc_queue"):
            getattr(L, name).argtypes = [vp, vp, u64]
        L.orc_load_tracks.argtypes = [vp, u32, vp, u64]
        L.orc_live.restype = u64
        L.orc_live.argtypes = [vp, u32]
        L.orc_read_tracks.argtypes = [vp, u32, vp, u64, C.POINTER(u64)]
        L.orc_step.argtypes = [vp]
        L.orc_run.argtypes = [vp, u64, C.c_int]
        L.orc_run_batched.argtypes = [vp, u64]
        L.orc_get_result.argtypes = [vp, C.POINTER(_Result), vp]
        L.orc_reset_tallies.argtypes = [vp]
        L.orc_set_primary_index.argtypes = [vp, u64]
        L.orc_set_trace.argtypes = [vp, C.c_int]
        L.orc_trace_size.restype = u64
        L.orc_trace_size.argtypes = [vp]
        L.orc_read_trace.argtypes = [vp, vp]
        L.orc_philox4x32_10.argtypes = [vp, vp, vp]
        L.orc_philox_array.argtypes = [vp, vp, vp, u64]
        for name in ("orc_u01_array", "orc_lg_array", "orc_ex_array"):
            getattr(L, name).argtypes = [vp, vp, u64]
        L.orc_sincos2pi_array.argtypes = [vp, vp, vp, u64]
        L.orc_rotate_array.argtypes = [vp] * 6 + [u64]
        L.orc_lookup_array.argtypes = [C.POINTER(_Tables), u32, u32, u32, vp, vp, u64]
        _LIB = L
    return _LIB


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _tables_struct(tables):
    data = np.ascontiguousarray(tables.data, dtype=np.float32)
    physics = int(getattr(tables, "physics", 0))
    data_x = np.ascontiguousarray(tables.data_x, dtype=np.float32) if physics else None
    t = _Tables(tables.n_bins, tables.n_materials, tables.e_min, tables.e_max,
                float(tables.ln_e_min), float(tables.inv_dln), tables.e_cut,
                data.ctypes.data_as(C.POINTER(C.c_float)), physics,
                data_x.ctypes.data_as(C.POINTER(C.c_float)) if physics else None)
    return t, (data, data_x)


class math_fns:
    """Array front-ends of the oracle's elementary functions (rules R1, R3, M8-M10, T13, S27)."""

    @staticmethod
    def philox(ctr, key):
        c = np.ascontiguousarray(ctr, dtype=np.uint32)
        k = np.ascontiguousarray(key, dtype=np.uint32)
        out = np.zeros(4, dtype=np.uint32)
        lib().orc_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
        return out

    @staticmethod
    def philox_array(ctr, key):
        c = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
        k = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
        assert c.shape[0] == k.shape[0]
        out = np.zeros((c.shape[0], 4), dtype=np.uint32)
        lib().orc_philox_array(_ptr(c), _ptr(k), _ptr(out), c.shape[0])
        return out

    @staticmethod
    def _unary(fn, x, in_dtype):
        x = np.ascontiguousarray(x, dtype=in_dtype)
        out = np.empty(x.shape, dtype=np.float32)
        getattr(lib(), fn)(_ptr(x), _ptr(out), x.size)
        return out

    @staticmethod
    def u01(x):
        return math_fns._unary("orc_u01_array", x, np.uint32)

    @staticmethod
    def lg(x):
        return math_fns._unary("orc_lg_array", x, np.float32)

    @staticmethod
    def ex(x):
        return math_fns._unary("orc_ex_array", x, np.float32)

    @staticmethod
    def sincos2pi(u):
        u = np.ascontiguousarray(u, dtype=np.float32)
        s = np.empty_like(u)
        c = np.empty_like(u)
        lib().orc_sincos2pi_array(_ptr(u), _ptr(s), _ptr(c), u.size)
        return s, c

    @staticmethod
    def rotate(d, st, ct, sphi, cphi):
        d = np.ascontiguousarray(d, dtype=np.float32).reshape(-1, 3)
        arrs = [np.ascontiguousarray(np.broadcast_to(a, d.shape[0]), dtype=np.float32)
                for a in (st, ct, sphi, cphi)]
        out = np.empty_like(d)
        lib().orc_rotate_array(_ptr(d), *[_ptr(a) for a in arrs], _ptr(out), d.shape[0])
        return out

    @staticmethod
    def lookup(tables, mat, group, qty, E):
        t, keep = _tables_struct(tables)
        E = np.ascontiguousarray(E, dtype=np.float32)
        out = np.empty_like(E)
        lib().orc_lookup_array(C.byref(t), mat, group, qty, _ptr(E), _ptr(out), E.size)
        del keep
        return out


class Oracle:
    """One oracle context: geometry + tables + seed, three track lists."""

    def __init__(self, geometry, tables, seed: int = 0):
        self._L = lib()
        g = _Geometry(geometry.n_layers, geometry.abs_mm, geometry.gap_mm, geometry.half_xy_mm,
                      geometry.mat_abs, geometry.mat_gap)
        t, keep = _tables_struct(tables)
        self._h = self._L.orc_create(C.byref(g), C.byref(t), seed)
        del keep
        if not self._h:
            raise ValueError("orc_create rejected its arguments")
        self.n_slabs = 2 * geometry.n_layers

    def close(self):
        if self._h:
            self._L.orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def inject(self, primaries: np.ndarray):
        p = np.ascontiguousarray(primaries)
        assert p.dtype.itemsize == 32
        if self._L.orc_inject(self._h, _ptr(p), p.shape[0]) != 0:
            raise ValueError("orc_inject: invalid primary")

    def set_primary_index(self, next_index: int):
        """Rule R4: global index of the next injected primary (event sharding)."""
        self._L.orc_set_primary_index(self._h, next_index)

    def queue(self, primaries: np.ndarray):
        p = np.ascontiguousarray(primaries)
        assert p.dtype.itemsize == 32
        self._L.orc_queue(self._h, _ptr(p), p.shape[0])

    def load_tracks(self, kind: int, tracks: np.ndarray):
        t = np.ascontiguousarray(tracks)
        assert t.dtype.itemsize == 56
        if self._L.orc_load_tracks(self._h, kind, _ptr(t), t.shape[0]) != 0:
            raise ValueError("orc_load_tracks")

    def live(self, kind: int) -> int:
        return int(self._L.orc_live(self._h, kind))

    def read_tracks(self, kind: int, dtype) -> np.ndarray:
        n = self.live(kind)
        out = np.zeros(n, dtype=dtype)
        m = C.c_uint64(0)
        rc = self._L.orc_read_tracks(self._h, kind, _ptr(out), n, C.byref(m))
        assert rc == 0 and m.value == n
        return out

    def step(self):
        self._L.orc_step(self._h)

    def run(self, max_iterations: int = 0, depth_first: bool = False):
        self._L.orc_run(self._h, max_iterations, 1 if depth_first else 0)

    def run_batched(self, batch: int):
        if self._L.orc_run_batched(self._h, batch) != 0:
            raise ValueError("orc_run_batched: invalid primary")

    def result(self) -> dict:
        r = _Result()
        edep = np.zeros(self.n_slabs, dtype=np.float64)
        self._L.orc_get_result(self._h, C.byref(r), _ptr(edep))
        out = {k: np.array(getattr(r, k), dtype=np.uint64) for k in
               ("live", "steps", "secondaries", "killed", "escaped_n", "slots_used")}
        out.update(iterations=int(r.iterations), e_injected=float(r.e_injected),
                   e_escaped=float(r.e_escaped), edep_slab=edep,
                   e_escaped_kind=np.array(r.e_escaped_kind, dtype=np.float64),
                   edep_layer=edep[0::2] + edep[1::2])
        return out

    def reset_tallies(self):
        self._L.orc_reset_tallies(self._h)

    def set_trace(self, on: bool):
        self._L.orc_set_trace(self._h, 1 if on else 0)

    def trace(self) -> np.ndarray:
        n = int(self._L.orc_trace_size(self._h))
        out = np.zeros(n, dtype=TRACE_DTYPE)
        self._L.orc_read_trace(self._h, _ptr(out))
        return out
