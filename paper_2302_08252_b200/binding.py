"""ctypes binding of include/adept.h — argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used here for device memory
(the workspace is a `torch.uint8` tensor the caller could equally allocate itself) and the stream.
Function names are the C names without the `adept_` prefix.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.environ.get("ADEPT_B200_LIB") or os.path.join(_HERE, "libadept_b200.so")

ADEPT_AOS, ADEPT_SOA, ADEPT_AOSOA32, ADEPT_AOSOA64, ADEPT_SOA16, ADEPT_AOSOA16, ADEPT_AOSOA128, ADEPT_HC16, ADEPT_AOSOA8 = 0, 1, 2, 3, 4, 5, 6, 7, 8
ADEPT_SPARSE_SINGLE, ADEPT_DENSE_DOUBLE = 0, 1
LAYOUTS = {"aos": ADEPT_AOS, "soa": ADEPT_SOA, "aosoa32": ADEPT_AOSOA32, "aosoa64": ADEPT_AOSOA64,
           "soa16": ADEPT_SOA16, "aosoa16": ADEPT_AOSOA16, "aosoa128": ADEPT_AOSOA128, "hc16": ADEPT_HC16, "aosoa8": ADEPT_AOSOA8}
SCHEMES = {"sparse": ADEPT_SPARSE_SINGLE, "dense": ADEPT_DENSE_DOUBLE}
FIELD_NAMES = ("pos.x", "pos.y", "pos.z", "dir.x", "dir.y", "dir.z", "ekin", "nial.0", "nial.1", "nial.2",
               "vol", "id_lo", "id_hi", "step")
STATUS = {0: "ADEPT_OK", -1: "ADEPT_EINVAL", -2: "ADEPT_ECAPACITY", -3: "ADEPT_ECUDA", -4: "ADEPT_ESTATE"}

TRACK_DTYPE = np.dtype([("pos", "<f4", (3,)), ("dir", "<f4", (3,)), ("ekin", "<f4"), ("nial", "<f4", (3,)),
                        ("vol", "<u4"), ("id_lo", "<u4"), ("id_hi", "<u4"), ("step", "<u4")])
PRIMARY_DTYPE = np.dtype([("kind", "<u4"), ("pos", "<f4", (3,)), ("dir", "<f4", (3,)), ("ekin", "<f4")])


class AdeptError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("%s: %s" % (STATUS.get(code, code), msg))
        self.code = code


class _Geometry(C.Structure):
    _fields_ = [("n_layers", C.c_uint32), ("abs_mm", C.c_float), ("gap_mm", C.c_float),
                ("half_xy_mm", C.c_float), ("mat_abs", C.c_uint32), ("mat_gap", C.c_uint32)]


class _Tables(C.Structure):
    _fields_ = [("n_bins", C.c_uint32), ("n_materials", C.c_uint32), ("e_min", C.c_float), ("e_max", C.c_float),
                ("ln_e_min", C.c_float), ("inv_dln", C.c_float), ("e_cut", C.c_float),
                ("data", C.POINTER(C.c_float)), ("physics", C.c_uint32), ("data_x", C.POINTER(C.c_float))]


class _Config(C.Structure):
    _fields_ = [("layout", C.c_int32), ("scheme", C.c_int32), ("capacity_per_kind", C.c_uint32),
                ("batch_primaries", C.c_uint32), ("seed", C.c_uint64), ("workspace", C.c_void_p),
                ("workspace_bytes", C.c_size_t), ("cuda_stream", C.c_void_p), ("instrument", C.c_uint32),
                ("flags", C.c_uint32)]


class _Counts(C.Structure):
    _fields_ = [("live", C.c_uint64 * 3), ("steps", C.c_uint64 * 3), ("secondaries", C.c_uint64 * 3),
                ("killed", C.c_uint64 * 3), ("escaped_n", C.c_uint64 * 3), ("slots_used", C.c_uint64 * 3),
                ("iterations", C.c_uint64), ("overflow", C.c_uint32), ("reserved", C.c_uint32)]


class _Result(C.Structure):
    _fields_ = [("total", _Counts), ("e_injected", C.c_double), ("e_escaped", C.c_double),
                ("edep_slab", C.POINTER(C.c_double)), ("edep_layer", C.POINTER(C.c_double))]


_SO_TIMING = os.path.join(_HERE, "libadept_b200_timing.so")   # -DADEPT_TIMING_SECTIONS variant (adept.h)
_LIBS: dict = {}


def lib(variant: str | None = None):
    """Load the C-ABI library (`variant="timing"`: the section-clock build of the same sources).
    Raises if it has not been built: there is no fallback path."""
    so = _SO_TIMING if variant == "timing" else _SO
    if so not in _LIBS:
        if not os.path.exists(so):
            raise ImportError("%s is missing: run `python -m paper_2302_08252_b200.build` (or "
                              "__graft_entry__.build()); there is no CPU fallback" % so)
        L = C.CDLL(so)
        vp, u64, u32 = C.c_void_p, C.c_uint64, C.c_uint32
        L.adept_workspace_bytes.restype = C.c_size_t
        L.adept_workspace_bytes.argtypes = [C.POINTER(_Geometry), C.POINTER(_Tables), C.POINTER(_Config)]
        L.adept_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Tables), C.POINTER(_Config), C.POINTER(vp)]
        L.adept_inject.argtypes = [vp, vp, u64]
        L.adept_set_primary_index.argtypes = [vp, u64]
        L.adept_step.argtypes = [vp, C.POINTER(_Counts)]
        L.adept_run.argtypes = [vp, u64, C.POINTER(_Result)]
        L.adept_get_result.argtypes = [vp, C.POINTER(_Result)]
        L.adept_load_tracks.argtypes = [vp, u32, vp, u64, vp]
        L.adept_read_tracks.argtypes = [vp, u32, vp, u64, C.POINTER(u64)]
        L.adept_read_counters.argtypes = [vp, vp, vp, vp]
        L.adept_instr_lines.restype = u64
        L.adept_instr_lines.argtypes = [vp]
        L.adept_instr_slots.restype = u64
        L.adept_instr_slots.argtypes = [vp]
        L.adept_field_offset.restype = u64
        L.adept_field_offset.argtypes = [C.c_int32, u32, u32, u32]
        L.adept_field_offset_kind.restype = u64
        L.adept_field_offset_kind.argtypes = [C.c_int32, u32, u32, u32, u32]
        L.adept_reset.argtypes = [vp]
        L.adept_destroy.argtypes = [vp]
        L.adept_last_error.restype = C.c_char_p
        L.adept_last_error.argtypes = [vp]
        L.adept_dev_math.argtypes = [C.c_int, vp, vp, u64, vp]
        L.adept_launch_index.restype = u32
        L.adept_launch_index.argtypes = [vp]
        L.adept_set_launch_index.argtypes = [vp, u32]
        L.adept_timing_sections.restype = C.c_int
        L.adept_timing_sections.argtypes = []
        L.adept_read_sections.argtypes = [vp, vp]
        L.adept_step_static.argtypes = [C.POINTER(_Geometry), C.POINTER(_Tables), C.POINTER(vp), C.POINTER(u32),
                                        C.POINTER(vp), u32, u32, vp, C.POINTER(_Result)]
        L.adept_step_static_bytes.restype = C.c_size_t
        L.adept_step_static_bytes.argtypes = []
        L.adept_step_static_error.restype = C.c_char_p
        L.adept_step_static_error.argtypes = []
        _LIBS[so] = L
    return _LIBS[so]


def field_offset(layout: int, capacity: int, slot: int, field: int, kind: int | None = None) -> int:
    if kind is not None:
        return int(lib().adept_field_offset_kind(layout, kind, capacity, slot, field))
    return int(lib().adept_field_offset(layout, capacity, slot, field))


def _counts_dict(c: _Counts) -> dict:
    d = {k: np.array(getattr(c, k), dtype=np.uint64) for k in
         ("live", "steps", "secondaries", "killed", "escaped_n", "slots_used")}
    d["iterations"] = int(c.iterations)
    d["overflow"] = int(c.overflow)
    return d


def dev_math(fn: int, inp, out_dtype, out_shape):
    """adept_dev_math on torch CUDA tensors (bit-equality tests of the elementary functions)."""
    import torch
    n = inp.shape[0]
    out = torch.empty(out_shape, dtype=out_dtype, device=inp.device)
    rc = lib().adept_dev_math(fn, inp.data_ptr(), out.data_ptr(), n, torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise AdeptError(rc, "adept_dev_math")
    torch.cuda.synchronize()
    return out


STATIC_MAX_TRACKS, STATIC_MAX_LAYERS, STATIC_MAX_BINS, STATIC_MAX_MATERIALS = 8192, 64, 256, 2


def step_static(geometry, tables, tracks_in, tracks_out, n_in, iterations: int = 1, stream=None):
    """adept_step_static: the transport step for callers that may not allocate device memory (a host that
    froze its memory plan, a hook that only gets buffers and a stream).  This wrapper allocates nothing on
    the device either: `tracks_in` / `tracks_out` are three existing torch CUDA uint8 tensors each (56-byte
    adept_track records; an input may be None when its count is 0), `n_in` the three input counts.
    Returns the counts / tallies dict of these iterations; `live[k]` records of tracks_out[k] are valid.
    Problems beyond the STATIC_MAX_* limits are refused by the library (AdeptError, ADEPT_EINVAL)."""
    import torch
    L = lib()
    g = _Geometry(geometry.n_layers, geometry.abs_mm, geometry.gap_mm, geometry.half_xy_mm,
                  geometry.mat_abs, geometry.mat_gap)
    data = np.ascontiguousarray(tables.data, dtype=np.float32)
    t = _Tables(tables.n_bins, tables.n_materials, tables.e_min, tables.e_max, float(tables.ln_e_min),
                float(tables.inv_dln), tables.e_cut, data.ctypes.data_as(C.POINTER(C.c_float)),
                int(getattr(tables, "physics", 0)), None)
    ins = (C.c_void_p * 3)(*[x.data_ptr() if x is not None else None for x in tracks_in])
    outs = (C.c_void_p * 3)(*[x.data_ptr() for x in tracks_out])
    out_cap = min(x.numel() * x.element_size() for x in tracks_out) // 56
    n = (C.c_uint32 * 3)(*[int(v) for v in n_in])
    r = _Result()
    slab = np.zeros(2 * geometry.n_layers, dtype=np.float64)
    layer = np.zeros(geometry.n_layers, dtype=np.float64)
    r.edep_slab = slab.ctypes.data_as(C.POINTER(C.c_double))
    r.edep_layer = layer.ctypes.data_as(C.POINTER(C.c_double))
    s = stream if stream is not None else torch.cuda.current_stream(tracks_out[0].device)
    rc = L.adept_step_static(C.byref(g), C.byref(t), ins, n, outs, out_cap, iterations, s.cuda_stream, C.byref(r))
    if rc != 0:
        raise AdeptError(rc, L.adept_step_static_error().decode())
    d = _counts_dict(r.total)
    d.update(e_escaped=float(r.e_escaped), edep_slab=slab, edep_layer=layer)
    return d


class Context:
    """adept_create ... adept_destroy.  `geometry`/`tables` are the workloads.* objects (plain data)."""

    def __init__(self, geometry, tables, *, layout="soa", scheme="dense", capacity, seed=0,
                 batch_primaries=0, instrument=False, device="cuda:0", stream=None, variant=None, flags=0):
        import torch
        self._L = lib(variant)
        self._torch = torch
        self.layout = LAYOUTS[layout] if isinstance(layout, str) else int(layout)
        self.scheme = SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
        self.n_layers = geometry.n_layers
        self._g = _Geometry(geometry.n_layers, geometry.abs_mm, geometry.gap_mm, geometry.half_xy_mm,
                            geometry.mat_abs, geometry.mat_gap)
        data = np.ascontiguousarray(tables.data, dtype=np.float32)
        physics = int(getattr(tables, "physics", 0))
        data_x = np.ascontiguousarray(tables.data_x, dtype=np.float32) if physics else None
        self._t = _Tables(tables.n_bins, tables.n_materials, tables.e_min, tables.e_max, float(tables.ln_e_min),
                          float(tables.inv_dln), tables.e_cut, data.ctypes.data_as(C.POINTER(C.c_float)), physics,
                          data_x.ctypes.data_as(C.POINTER(C.c_float)) if physics else None)
        cfg = _Config(self.layout, self.scheme, capacity, batch_primaries, seed, None, 0, None,
                      1 if instrument else 0, flags)
        nbytes = self._L.adept_workspace_bytes(C.byref(self._g), C.byref(self._t), C.byref(cfg))
        if nbytes == 0:
            raise AdeptError(-1, "adept_workspace_bytes rejected the arguments")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        cfg.workspace = self.workspace.data_ptr()
        cfg.workspace_bytes = nbytes
        cfg.cuda_stream = self.stream.cuda_stream
        self._h = C.c_void_p()
        rc = self._L.adept_create(C.byref(self._g), C.byref(self._t), C.byref(cfg), C.byref(self._h))
        if rc != 0:
            raise AdeptError(rc, self._L.adept_last_error(None).decode())
        self.capacity = capacity
        self.instrument = bool(instrument)

    # -- plumbing -------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != 0:
            raise AdeptError(rc, self._L.adept_last_error(self._h).decode())

    def destroy(self):
        if getattr(self, "_h", None):
            self._L.adept_destroy(self._h)
            self._h = None

    close = destroy

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- the ABI, one method per call -----------------------------------------------------------
    def inject(self, primaries: np.ndarray):
        p = np.ascontiguousarray(primaries)
        assert p.dtype.itemsize == 32
        self._check(self._L.adept_inject(self._h, p.ctypes.data, p.shape[0]))

    def set_primary_index(self, next_index: int):
        self._check(self._L.adept_set_primary_index(self._h, next_index))

    def step(self, sync: bool = True):
        if not sync:
            self._check(self._L.adept_step(self._h, None))
            return None
        c = _Counts()
        self._check(self._L.adept_step(self._h, C.byref(c)))
        return _counts_dict(c)

    def _result(self, fn, *args):
        r = _Result()
        slab = np.zeros(2 * self.n_layers, dtype=np.float64)
        layer = np.zeros(self.n_layers, dtype=np.float64)
        r.edep_slab = slab.ctypes.data_as(C.POINTER(C.c_double))
        r.edep_layer = layer.ctypes.data_as(C.POINTER(C.c_double))
        self._check(fn(self._h, *args, C.byref(r)))
        d = _counts_dict(r.total)
        d.update(e_injected=float(r.e_injected), e_escaped=float(r.e_escaped), edep_slab=slab, edep_layer=layer)
        return d

    def run(self, max_iterations: int = 0):
        return self._result(self._L.adept_run, max_iterations)

    def result(self):
        return self._result(self._L.adept_get_result)

    def load_tracks(self, kind: int, tracks: np.ndarray, slots: np.ndarray | None = None):
        t = np.ascontiguousarray(tracks)
        assert t.dtype.itemsize == 56
        s = None
        if slots is not None:
            s = np.ascontiguousarray(slots, dtype=np.uint32)
            assert s.shape[0] == t.shape[0]
        self._check(self._L.adept_load_tracks(self._h, kind, t.ctypes.data, t.shape[0],
                                              s.ctypes.data if s is not None else None))

    def read_tracks(self, kind: int, cap: int | None = None, out: np.ndarray | None = None):
        """Without `out`: returns a new array of the live tracks.  With `out` (a TRACK_DTYPE host array,
        e.g. pinned): fills it in place and returns the number of tracks."""
        n = C.c_uint64(0)
        if out is not None:
            assert out.dtype.itemsize == 56 and out.flags["C_CONTIGUOUS"]
            self._check(self._L.adept_read_tracks(self._h, kind, out.ctypes.data, out.shape[0], C.byref(n)))
            return int(n.value)
        cap = (self.capacity + 127) // 128 * 128 if cap is None else cap    # the library rounds capacity up to whole tiles
        buf = np.empty(cap, dtype=TRACK_DTYPE)
        self._check(self._L.adept_read_tracks(self._h, kind, buf.ctypes.data, cap, C.byref(n)))
        return buf[: n.value].copy()

    def read_counters(self):
        n_lines = int(self._L.adept_instr_lines(self._h))
        n_slots = int(self._L.adept_instr_slots(self._h))
        rw = np.zeros((3, 14, 2), dtype=np.uint64)
        lines = np.zeros((3, n_lines), dtype=np.uint32)
        slots = np.zeros((3, n_slots), dtype=np.uint32)
        self._check(self._L.adept_read_counters(self._h, rw.ctypes.data, lines.ctypes.data, slots.ctypes.data))
        return dict(field_rw=rw, lines=lines, slots=slots)

    def launch_index(self) -> int:
        return int(self._L.adept_launch_index(self._h))

    def set_launch_index(self, index: int):
        self._check(self._L.adept_set_launch_index(self._h, index))

    def snapshot(self):
        """(workspace copy, launch index): what `rewind` needs (adept.h "Workspace").  No call may be in flight."""
        return self.workspace.clone(), int(self._L.adept_launch_index(self._h))

    def rewind(self, snap):
        self.workspace.copy_(snap[0])
        self._check(self._L.adept_set_launch_index(self._h, snap[1]))

    def read_sections(self):
        """Timing variant: warp-cycles per kernel section (adept.h adept_read_sections)."""
        out = np.zeros(8, dtype=np.uint64)
        self._check(self._L.adept_read_sections(self._h, out.ctypes.data))
        return out

    def reset(self):
        self._check(self._L.adept_reset(self._h))
