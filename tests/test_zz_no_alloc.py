"""adept_step_static -- the transport step for callers that are not allowed to allocate -- against the
ordinary path (adept_create on a caller-allocated workspace, adept_load_tracks, adept_step,
adept_read_tracks), on the same seeded tracks.

Why the entry point exists: a host that reserved all device memory at start-up, a plugin hook that only
receives buffers and a stream, or code that cannot afford the device-wide synchronisation of
cudaMalloc / cudaFree cannot create an adept context (workspace, pinned buffer, stream, events).
adept_step_static keeps what the workspace would hold in one fixed __device__ array of the library
(about 2.7 MiB per GPU), so it is limited to 8192 tracks per kind, 64 layers, 256 bins, 2 materials and
the basic physics, and all calls share that array.

What is checked: both paths run the same kernel, so every word of every track (sorted by id), every
count and every fixed-point tally must be EQUAL, not merely within the 1e-5 / 1e-4 tolerances of
test_gpu_parity.py.  Two calls are made in a row with different populations and iteration counts: the
second must not see anything the first left in the shared array.

This file is collected last on purpose (pytest -x would otherwise hide later tests behind a failure
here) and passes alone in a fresh process as well as after the rest of the suite."""
import numpy as np
import pytest

from workloads import CONFIGS, TRACK_DTYPE, gen_tracks, geometry_for, tables_for
from tests.helpers import sort_by_id

COUNT_KEYS = ("live", "steps", "secondaries", "killed", "escaped_n", "slots_used")
CAPACITY = 8192   # ADEPT_STATIC_MAX_TRACKS


def _existing_path(geo, tab, tracks, iterations):
    """adept_create / load_tracks / step / read_tracks on a torch-allocated workspace."""
    from paper_2302_08252_b200 import Context
    ctx = Context(geo, tab, layout="aosoa32", scheme="dense", capacity=CAPACITY, seed=0)
    for k in range(3):
        if tracks[k].shape[0]:
            ctx.load_tracks(k, tracks[k])
    for _ in range(iterations):
        ctx.step()
    res = ctx.result()
    out = [ctx.read_tracks(k) for k in range(3)]
    ctx.destroy()
    return res, out


def _static_path(geo, tab, tracks, iterations, d_in, d_out):
    """adept_step_static on device buffers that exist already (d_in / d_out are reused between calls)."""
    import torch
    from paper_2302_08252_b200.binding import step_static
    for k in range(3):
        raw = torch.from_numpy(np.ascontiguousarray(tracks[k]).view(np.uint8))
        d_in[k][: raw.numel()].copy_(raw)
        d_out[k].fill_(0xEE)   # stale output must not pass for a result
    res = step_static(geo, tab, d_in, d_out, [t.shape[0] for t in tracks], iterations=iterations)
    torch.cuda.synchronize()
    out = [d_out[k].cpu().numpy().view(TRACK_DTYPE)[: int(res["live"][k])].copy() for k in range(3)]
    return res, out


def _assert_same(a, b, what):
    (ra, ta), (rb, tb) = a, b
    for key in COUNT_KEYS:
        assert (np.asarray(ra[key]) == np.asarray(rb[key])).all(), "%s: %s static %s existing %s" % (what, key, ra[key], rb[key])
    assert ra["iterations"] == rb["iterations"] and ra["overflow"] == rb["overflow"] == 0, what
    assert (ra["edep_slab"] == rb["edep_slab"]).all(), "%s: per-slab energy deposit differs" % what
    assert (ra["edep_layer"] == rb["edep_layer"]).all() and ra["e_escaped"] == rb["e_escaped"], what
    for k in range(3):
        assert ta[k].shape[0] == tb[k].shape[0], "%s: kind %d has %d vs %d tracks" % (what, k, ta[k].shape[0], tb[k].shape[0])
        x = sort_by_id(ta[k]).view(np.uint32).reshape(-1, 14)
        y = sort_by_id(tb[k]).view(np.uint32).reshape(-1, 14)
        assert (x == y).all(), "%s: kind %d, %d track words differ" % (what, k, int((x != y).sum()))


@pytest.mark.gpu
def test_step_static_equals_the_workspace_path_on_two_calls_in_a_row():
    import torch
    c = CONFIGS["single_step"]
    geo, tab = geometry_for("single_step"), tables_for("single_step")
    d_in = [torch.empty(CAPACITY * 56, dtype=torch.uint8, device="cuda:0") for _ in range(3)]
    d_out = [torch.empty(CAPACITY * 56, dtype=torch.uint8, device="cuda:0") for _ in range(3)]
    # call 1: 6000 tracks (2400 e-, 600 e+, 3000 gamma: 47 tiles and ragged tails), one iteration;
    # call 2: a smaller, different population for three iterations -- counters, tallies and the record
    # arrays the first call left behind in the library's array must not show
    cases = ((6000, c["seed"], 1), (1777, c["seed"] + 100, 3))
    before = torch.cuda.memory_allocated()
    got = []
    for n, seed, iterations in cases:
        tracks = gen_tracks(n, seed, geo, c["e_max"], c["fractions"])
        got.append((tracks, iterations, _static_path(geo, tab, tracks, iterations, d_in, d_out)))
    assert torch.cuda.memory_allocated() == before, "the wrapper of the no-allocation entry point allocated device memory"
    for i, (tracks, iterations, static) in enumerate(got):
        existing = _existing_path(geo, tab, tracks, iterations)
        assert sum(int(v) for v in static[0]["secondaries"]) > 0 and sum(int(v) for v in static[0]["killed"]) > 0
        _assert_same(static, existing, "call %d" % (i + 1))
    assert (got[0][2][0]["steps"] != got[1][2][0]["steps"]).any()


@pytest.mark.gpu
def test_step_static_runs_a_whole_small_shower():
    """Config 1 (16 primaries of 10 MeV, 4 layers, 64 bins) fits the fixed array: all of its iterations in
    one call, against adept_run's tallies."""
    import torch
    from paper_2302_08252_b200 import Context
    from workloads import gen_primaries
    c = CONFIGS["tiny"]
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    ctx = Context(geo, tab, layout="aosoa32", scheme="dense", capacity=c["capacity"], seed=c["seed"])
    ctx.inject(gen_primaries(c["n_primaries"], c["e_primary"]))
    start = [ctx.read_tracks(k) for k in range(3)]
    ref = ctx.run()
    ctx.destroy()
    d_in = [torch.empty(CAPACITY * 56, dtype=torch.uint8, device="cuda:0") for _ in range(3)]
    d_out = [torch.empty(CAPACITY * 56, dtype=torch.uint8, device="cuda:0") for _ in range(3)]
    res, out = _static_path(geo, tab, start, 200, d_in, d_out)
    assert ref["iterations"] < 200 and res["iterations"] == ref["iterations"]   # idle launches are not counted
    assert all(o.shape[0] == 0 for o in out)
    for key in ("steps", "secondaries", "killed", "escaped_n"):
        assert (res[key] == ref[key]).all(), key
    assert (res["edep_slab"] == ref["edep_slab"]).all() and res["e_escaped"] == ref["e_escaped"]


def test_step_static_refuses_what_does_not_fit_its_array():
    """Argument checks come before any CUDA call (they run without a GPU): sizes beyond the fixed array
    are an error with a message that names the limit, never a truncated run."""
    import ctypes as C
    from paper_2302_08252_b200 import binding as B
    L = B.lib()
    assert 2_000_000 < L.adept_step_static_bytes() < 4 * 1024 * 1024   # "modest": what every GPU holds until exit
    data = np.zeros(2 * 2 * 3 * 257, dtype=np.float32)

    def call(n_layers=50, n_bins=256, n_mat=2, physics=0, n0=16, iterations=1):
        g = B._Geometry(n_layers, 2.3, 5.7, 200.0, 0, 1)
        t = B._Tables(n_bins, n_mat, 0.1, 1e4, 0.0, 1.0, 0.1, data.ctypes.data_as(C.POINTER(C.c_float)), physics, None)
        ptrs = (C.c_void_p * 3)(256, 256, 256)   # never dereferenced: the checks fail first
        n = (C.c_uint32 * 3)(n0, 0, 0)
        r = B._Result()
        rc = L.adept_step_static(C.byref(g), C.byref(t), ptrs, n, ptrs, 0, iterations, None, C.byref(r))
        return rc, L.adept_step_static_error().decode()

    for kw, word in ((dict(n0=B.STATIC_MAX_TRACKS + 1), "ADEPT_STATIC_MAX_TRACKS"), (dict(n_layers=B.STATIC_MAX_LAYERS + 1), "ADEPT_STATIC_MAX_LAYERS"),
                     (dict(n_bins=B.STATIC_MAX_BINS + 1), "ADEPT_STATIC_MAX_BINS"), (dict(n_mat=B.STATIC_MAX_MATERIALS + 1), "ADEPT_STATIC_MAX_MATERIALS"),
                     (dict(physics=1), "physics"), (dict(iterations=0), "iterations")):
        rc, msg = call(**kw)
        assert rc == -1 and word in msg, (kw, rc, msg)
