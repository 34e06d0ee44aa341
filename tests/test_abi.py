"""The C-ABI boundary without a GPU: the library loads, exports every function include/adept.h
declares, and its pure host arithmetic (workspace sizing, layout offsets, argument validation that
happens before any CUDA call) behaves as documented.  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2302_08252_b200 import build
    build.build_all()
    from paper_2302_08252_b200 import binding
    return binding


def declared_functions():
    text = open(os.path.join(ROOT, "include", "adept.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(adept_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_function(L):
    names = declared_functions()
    assert {"adept_create", "adept_inject", "adept_step", "adept_run"} <= set(names)   # north_star's four calls
    lib = L.lib()
    for n in names:
        assert hasattr(lib, n), "libadept_b200.so does not export %s" % n
    assert len(names) >= 20


def test_timing_variant_exports_the_same_abi(L):
    """libadept_b200_timing.so (section clocks, -DADEPT_TIMING_SECTIONS) is the same library."""
    lib, timing = L.lib(), L.lib("timing")
    for n in declared_functions():
        assert hasattr(timing, n), "libadept_b200_timing.so does not export %s" % n
    assert lib.adept_timing_sections() == 0 and timing.adept_timing_sections() == 1
    assert timing.adept_read_sections(None, None) == -1


def test_record_sizes_match_the_header(L):
    assert L.TRACK_DTYPE.itemsize == 56 and L.PRIMARY_DTYPE.itemsize == 32
    assert C.sizeof(L._Counts) == 8 * 19 + 8 and C.sizeof(L._Geometry) == 24


def _args(L, layout=1, scheme=1, capacity=4096, n_layers=50, n_bins=256, instrument=0):
    g = L._Geometry(n_layers, 2.3, 5.7, 200.0, 0, 1)
    t = L._Tables(n_bins, 2, 0.1, 1e4, 0.0, 1.0, 0.1, None, 0, None)
    c = L._Config(layout, scheme, capacity, 0, 0, None, 0, None, instrument, 0)
    return g, t, c


def test_workspace_bytes_is_host_arithmetic(L):
    lib = L.lib()
    size = lambda **k: lib.adept_workspace_bytes(*[C.byref(x) for x in _args(L, **k)])
    base = size()
    assert base > 3 * 2 * 4096 * 56                                  # three kinds, two dense arrays
    assert size(capacity=8192) > base and size(capacity=4097) == size(capacity=4224)   # rounded to 128 slots (one tile)
    assert size(layout=0) > size(layout=1) == size(layout=2) == size(layout=3) == size(layout=4) == size(layout=7) == size(layout=8)   # AoS records are padded to 64 B
    assert size(scheme=0) < base                                     # one slot array + two slot lists
    assert size(instrument=1) > base
    for bad in (dict(layout=9), dict(scheme=5), dict(capacity=0), dict(n_layers=0), dict(n_bins=0)):
        assert size(**bad) == 0


def test_workspace_bytes_with_extended_physics_and_flags(L):
    """physics 2 adds the side arrays of the three multiple-scattering words (e-, e+; per buffer), slot
    recycling the free rings; the extended physics is refused with instrumentation or recycling."""
    lib = L.lib()

    def size(physics=0, flags=0, instrument=0, scheme=1, capacity=4096):
        g, t, c = _args(L, scheme=scheme, capacity=capacity, instrument=instrument)
        t.physics = physics
        c.flags = flags
        return lib.adept_workspace_bytes(C.byref(g), C.byref(t), C.byref(c))

    base_d, base_s = size(), size(scheme=0)
    nodes = 257
    assert abs((size(physics=1) - base_d) - 2 * nodes * 16) < 256          # a third table group (e+ extras), blocks are 256-byte aligned
    assert size(physics=2) - size(physics=1) == 2 * 2 * 3 * 4096 * 4       # 2 kinds x 2 buffers x 3 words
    assert size(physics=2, scheme=0) - size(physics=1, scheme=0) == 2 * 1 * 3 * 4096 * 4
    assert size(scheme=0, flags=1) - base_s == 3 * 4096 * 4                # one ring per kind
    assert size(flags=1) == base_d                                          # the dense scheme ignores the flag
    for bad in (dict(physics=3), dict(physics=1, instrument=1), dict(physics=2, scheme=0, flags=1), dict(flags=2)):
        assert size(**bad) == 0


def test_field_offset_follows_the_three_mappings(L):
    cap = 4096
    for slot in (0, 1, 31, 32, 33, 1000, 4095):
        for f in range(14):
            assert L.field_offset(L.ADEPT_AOS, cap, slot, f) == 4 * (slot * 16 + f)       # 64-byte records
            assert L.field_offset(L.ADEPT_SOA, cap, slot, f) == 4 * (f * cap + slot)       # 14 arrays
            assert L.field_offset(L.ADEPT_AOSOA32, cap, slot, f) == 4 * ((slot // 32) * 448 + f * 32 + slot % 32)
            assert L.field_offset(L.ADEPT_AOSOA64, cap, slot, f) == 4 * ((slot // 64) * 896 + f * 64 + slot % 64)
            for lay, n in ((5, 16), (6, 128), (8, 8)):                                    # more AoSoA lane counts
                assert L.field_offset(lay, cap, slot, f) == 4 * ((slot // n) * 14 * n + f * n + slot % n)
            want = (f // 4) * 16 * cap + slot * 16 + (f % 4) * 4 if f < 12 else 48 * cap + slot * 8 + (f - 12) * 4
            assert L.field_offset(L.ADEPT_SOA16, cap, slot, f) == want          # 16-byte field groups
    assert L.field_offset(L.ADEPT_SOA, cap, 0, 14) == 2**64 - 1 and L.field_offset(9, cap, 0, 0) == 2**64 - 1
    # HC16: the SoA16 geometry with the words regrouped per particle kind (hot {pos, step}, hot
    # {nial.., vol} / {ekin, nial.0-1, vol}, read-mostly {dir, ekin} / {dir, nial.2}, cold ids)
    order = {2: ["pos.x", "pos.y", "pos.z", "step", "nial.0", "nial.1", "nial.2", "vol", "dir.x", "dir.y", "dir.z", "ekin", "id_lo", "id_hi"],
             0: ["pos.x", "pos.y", "pos.z", "step", "ekin", "nial.0", "nial.1", "vol", "dir.x", "dir.y", "dir.z", "nial.2", "id_lo", "id_hi"]}
    order[1] = order[0]
    assert L.field_offset(L.ADEPT_HC16, cap, 0, 0) == 2**64 - 1                  # needs the kind
    for kind in range(3):
        for slot in (0, 5, 4095):
            for f, name in enumerate(L.FIELD_NAMES):
                pos = order[kind].index(name)
                assert L.field_offset(L.ADEPT_HC16, cap, slot, f, kind=kind) == L.field_offset(L.ADEPT_SOA16, cap, slot, pos)
        assert L.field_offset(L.ADEPT_SOA, cap, 3, 2, kind=kind) == L.field_offset(L.ADEPT_SOA, cap, 3, 2)
    assert L.field_offset(L.ADEPT_HC16, cap, 0, 0, kind=3) == 2**64 - 1
    # every (slot, field) has its own word in every layout
    for lay, words in ((L.ADEPT_AOS, 16), (L.ADEPT_SOA, 14), (L.ADEPT_AOSOA32, 14), (L.ADEPT_AOSOA64, 14),
                       (L.ADEPT_SOA16, 14)):
        offs = {L.field_offset(lay, 128, s, f) for s in range(128) for f in range(14)}
        assert len(offs) == 128 * 14 and max(offs) < 128 * words * 4


def test_create_rejects_bad_arguments_before_touching_the_device(L):
    lib = L.lib()
    g, t, c = _args(L)
    h = C.c_void_p()
    assert lib.adept_create(C.byref(g), C.byref(t), C.byref(c), C.byref(h)) == -1      # tables.data is NULL
    assert b"NULL" in lib.adept_last_error(None)
    data = np.zeros(2 * 2 * 3 * 257, dtype=np.float32)
    t.data = data.ctypes.data_as(C.POINTER(C.c_float))
    assert lib.adept_create(C.byref(g), C.byref(t), C.byref(c), C.byref(h)) == -1      # no workspace
    assert b"workspace" in lib.adept_last_error(None)
    assert lib.adept_create(C.byref(g), C.byref(t), C.byref(c), None) == -1
    assert not h.value
    for fn in ("adept_destroy", "adept_reset"):
        assert getattr(lib, fn)(None) == -1
    assert lib.adept_set_primary_index(None, 5) == -1
    assert lib.adept_dev_math(9, None, None, 0, None) == -1
