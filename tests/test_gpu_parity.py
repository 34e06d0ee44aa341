"""GPU parity: the CUDA library (through its C ABI) against the oracle, element by element on the
same seeded inputs.  Integer results (counts, ids, steps, slab indices) must be bit-exact; fp32
track fields within 1e-5 relative (they are in fact bit-exact, which the tests report); per-layer
energy deposit within 1e-4 relative (BASELINE.json north_star).  `-m gpu` only."""
import numpy as np
import pytest

from oracle import Oracle, math_fns
from workloads import CONFIGS, gen_primaries, gen_sweep, gen_tracks, geometry_for, tables_for
from tests.helpers import make_tracks, sort_by_id

pytestmark = pytest.mark.gpu

LAYOUTS = ("aos", "soa", "aosoa32", "aosoa64", "soa16", "aosoa16", "aosoa128", "hc16", "aosoa8")
SCHEMES = ("dense", "sparse")
INT_FIELDS = ("vol", "id_lo", "id_hi", "step")
F32_FIELDS = ("pos", "dir", "ekin", "nial")


def _ctx(*a, **k):
    from paper_2302_08252_b200 import Context
    return Context(*a, **k)


def compare_tracks(gpu, ref, what=""):
    """Per-track comparison after sorting by id.  Returns the number of fp32 words that differ in
    their last bits (reported, must be within 1e-5 relative)."""
    assert gpu.shape[0] == ref.shape[0], "%s: %d tracks vs oracle %d" % (what, gpu.shape[0], ref.shape[0])
    g, r = sort_by_id(gpu), sort_by_id(ref)
    for f in INT_FIELDS:
        assert (g[f] == r[f]).all(), "%s: integer field %s differs" % (what, f)
    inexact = 0
    for f in F32_FIELDS:
        a, b = g[f].astype(np.float64), r[f].astype(np.float64)
        inexact += int((g[f].view(np.uint32) != r[f].view(np.uint32)).sum())
        tol = 1e-5 * np.maximum(np.abs(b), 1e-30)
        assert (np.abs(a - b) <= tol).all(), "%s: fp32 field %s beyond 1e-5 relative" % (what, f)
    return inexact


def compare_counts(g, r, keys=("live", "steps", "secondaries", "killed", "escaped_n"), what=""):
    for k in keys:
        assert (np.asarray(g[k]) == np.asarray(r[k])).all(), "%s: %s gpu %s oracle %s" % (what, k, g[k], r[k])


# ------------------------------------------------------------------ elementary functions -----
def test_device_math_is_bit_equal_to_the_oracle():
    import torch
    from paper_2302_08252_b200 import dev_math
    rng = np.random.default_rng(11)
    ck = rng.integers(0, 2**32, size=(200000, 6), dtype=np.uint64).astype(np.uint32)
    out = dev_math(0, torch.from_numpy(ck.view(np.int32)).cuda(), torch.int32, (ck.shape[0], 4)).cpu().numpy().view(np.uint32)
    assert (out == math_fns.philox_array(ck[:, :4], ck[:, 4:])).all()
    x = (np.arange(0, 1 << 23, 3, dtype=np.uint64) << np.uint64(9)).astype(np.uint32)
    u = dev_math(1, torch.from_numpy(x.view(np.int32)).cuda(), torch.float32, (x.shape[0],)).cpu().numpy()
    assert (u.view(np.uint32) == math_fns.u01(x).view(np.uint32)).all()

    def sweep(lo, hi, stride):
        a, b = np.float32(lo).view(np.uint32), np.float32(hi).view(np.uint32)
        return np.arange(int(a), int(b), stride, dtype=np.uint32).view(np.float32)

    xs = np.concatenate([sweep(1e-8, 1e5, 7), u])
    y = dev_math(2, torch.from_numpy(xs).cuda(), torch.float32, (xs.shape[0],)).cpu().numpy()
    assert (y.view(np.uint32) == math_fns.lg(xs).view(np.uint32)).all()
    xs = np.concatenate([sweep(1e-6, 20.0, 11), -sweep(1e-6, 30.0, 11), np.float32([0.0])])
    y = dev_math(3, torch.from_numpy(xs).cuda(), torch.float32, (xs.shape[0],)).cpu().numpy()
    assert (y.view(np.uint32) == math_fns.ex(xs).view(np.uint32)).all()
    sc = dev_math(4, torch.from_numpy(u).cuda(), torch.float32, (u.shape[0], 2)).cpu().numpy()
    s, c = math_fns.sincos2pi(u)
    assert (sc[:, 0].view(np.uint32) == s.view(np.uint32)).all() and (sc[:, 1].view(np.uint32) == c.view(np.uint32)).all()


def test_inrange_division_is_the_ieee_quotient():
    """csrc/mathfn.cuh div_rn_inrange (the division inside lg, rule M8) against numpy's correctly
    rounded fp32 division, bit for bit, over its whole admitted operand range and on lg's operands."""
    import torch
    from paper_2302_08252_b200 import dev_math
    rng = np.random.default_rng(5)
    n = 4_000_000
    mant = lambda: (rng.integers(0, 1 << 23, n, dtype=np.uint64).astype(np.uint32) | np.uint32(0x3F800000)).view(np.float32)
    sign = lambda: np.where(rng.random(n) < 0.5, np.float32(-1), np.float32(1))
    a = np.ldexp(mant(), rng.integers(-100, 40, n)).astype(np.float32) * sign()
    b = np.ldexp(mant(), rng.integers(-60, 20, n)).astype(np.float32) * sign()
    m = (rng.integers(0, 1 << 23, n, dtype=np.uint64).astype(np.uint32) | np.uint32(0x3F800000)).view(np.float32)
    m = np.where(m > np.float32(1.41421354), m * np.float32(0.5), m)
    a = np.concatenate([a, m - np.float32(1), np.float32([0.0, 0.0, 1.0, -1.0])])
    b = np.concatenate([b, m + np.float32(1), np.float32([2.0, -3.0, 3.0, 3.0])])
    ab = np.stack([a, b], axis=1).astype(np.float32)
    q = dev_math(5, torch.from_numpy(ab).cuda(), torch.float32, (ab.shape[0],)).cpu().numpy()
    with np.errstate(all="ignore"):
        ref = (a / b).astype(np.float32)
    nz = ref != 0
    assert (q[nz].view(np.uint32) == ref[nz].view(np.uint32)).all()
    assert (q[~nz] == 0).all()


# ------------------------------------------------------------------------ single step --------
@pytest.fixture(scope="module")
def single_step_case():
    c = CONFIGS["single_step"]
    geo, tab = geometry_for("single_step"), tables_for("single_step")
    n = 200000 + 77                                  # several tiles per kind and a ragged tail
    pop = gen_tracks(n, c["seed"], geo, c["e_max"], c["fractions"])
    # make the step exercise every branch: some spent nial, some forced interactions, e+ at rest
    rng = np.random.default_rng(123)
    for k in range(3):
        t = pop[k]
        m = rng.random(t.shape[0])
        t["nial"][m < 0.10] = -1.0
        for j in range(3 if k == 2 else 1):
            t["nial"][(m >= 0.10 + 0.05 * j) & (m < 0.15 + 0.05 * j), j] = 1e-30
    pop[1]["ekin"][::7] = np.float32(0.05)
    o = Oracle(geo, tab, seed=c["seed"])
    for k in range(3):
        o.load_tracks(k, pop[k])
    o.step()
    ref = dict(result=o.result(), tracks=[o.read_tracks(k, pop[0].dtype) for k in range(3)])
    return geo, tab, pop, ref


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("layout", LAYOUTS)
def test_single_step_matches_oracle(single_step_case, layout, scheme):
    geo, tab, pop, ref = single_step_case
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=1 << 19, seed=3)
    for k in range(3):
        ctx.load_tracks(k, pop[k])
    counts = ctx.step()
    compare_counts(counts, ref["result"], what="%s/%s" % (layout, scheme))
    inexact = sum(compare_tracks(ctx.read_tracks(k), ref["tracks"][k], "%s/%s kind %d" % (layout, scheme, k))
                  for k in range(3))
    res = ctx.result()
    assert np.allclose(res["edep_slab"], ref["result"]["edep_slab"], rtol=1e-9, atol=1e-9)
    assert abs(res["e_escaped"] - ref["result"]["e_escaped"]) <= 1e-9 * max(1.0, ref["result"]["e_escaped"])
    print("single step %s/%s: %d fp32 words differ in the last bits" % (layout, scheme, inexact))
    assert inexact == 0          # rule M7: the arithmetic is reproducible bit for bit
    ctx.destroy()


# ------------------------------------------------------------------------ showers ------------
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("layout", LAYOUTS)
def test_tiny_shower_matches_oracle_every_iteration(layout, scheme):
    c = CONFIGS["tiny"]
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    prim = gen_primaries(c["n_primaries"], c["e_primary"])
    o = Oracle(geo, tab, seed=c["seed"])
    o.inject(prim)
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=c["capacity"], seed=c["seed"])
    ctx.inject(prim)
    it = 0
    while True:
        for k in range(3):
            compare_tracks(ctx.read_tracks(k), o.read_tracks(k, prim.dtype if False else make_tracks(1).dtype),
                           "iteration %d kind %d" % (it, k))
        if sum(o.live(k) for k in range(3)) == 0:
            break
        o.step()
        counts = ctx.step()
        compare_counts(counts, o.result(), what="iteration %d" % it)
        it += 1
    r, g = o.result(), ctx.result()
    assert g["iterations"] == r["iterations"] == it
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-12)
    assert abs(g["e_escaped"] - r["e_escaped"]) <= 1e-9 * max(1.0, r["e_escaped"])
    assert abs(g["edep_slab"].sum() + g["e_escaped"] - g["e_injected"]) < 1e-6 * g["e_injected"]
    if scheme == "dense":
        assert (g["slots_used"] == r["slots_used"]).all()
    else:   # rule S30: bump allocation, never recycled within a batch
        injected = np.array([c["n_primaries"], 0, 0], dtype=np.uint64)
        assert (g["slots_used"] == injected + r["secondaries"]).all()
    ctx.destroy()


@pytest.mark.parametrize("layout,scheme", [("soa", "dense"), ("aosoa32", "dense"), ("aosoa64", "dense"), ("soa16", "dense"),
                                           ("aos", "sparse")])
def test_full_showers_run_matches_oracle(layout, scheme):
    """Config 2 at reduced primaries (100 x 1 GeV) so that the oracle takes well under a second."""
    c = CONFIGS["full"]
    geo, tab = geometry_for("full"), tables_for("full")
    prim = gen_primaries(100, c["e_primary"])
    o = Oracle(geo, tab, seed=c["seed"])
    o.inject(prim)
    o.run()
    r = o.result()
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=1 << 19, seed=c["seed"])
    ctx.inject(prim)
    g = ctx.run()
    compare_counts(g, r)
    assert g["iterations"] == r["iterations"]
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-9)
    assert abs(g["e_escaped"] - r["e_escaped"]) <= 1e-9 * r["e_injected"]
    ctx.destroy()


def test_batched_run_matches_oracle():
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    prim = gen_primaries(25, 10.0)
    o = Oracle(geo, tab, seed=9)
    o.queue(prim)
    o.run_batched(5)
    r = o.result()
    for scheme in SCHEMES:
        ctx = _ctx(geo, tab, layout="soa", scheme=scheme, capacity=4096, seed=9, batch_primaries=5)
        ctx.inject(prim)
        g = ctx.run()
        compare_counts(g, r, what=scheme)
        assert g["iterations"] == r["iterations"]
        assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-12)
        if scheme == "dense":
            assert (g["slots_used"] == r["slots_used"]).all()
        ctx.destroy()


# -------------------------------------------------------------------- config 4 populations ---
@pytest.mark.parametrize("layout", LAYOUTS)
def test_sweep_population_sparse_slots_and_forced_secondaries(layout):
    geo, tab = geometry_for("sweep"), tables_for("sweep")
    span = 1 << 16
    pop = gen_sweep(0.3, span=span)
    o = Oracle(geo, tab, seed=4)
    for k in range(3):
        o.load_tracks(k, pop[k]["tracks"])
    o.step()
    r = o.result()
    forced = [int(p["forced"].sum()) for p in pop]
    for scheme in SCHEMES:
        ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=span + (1 << 14), seed=4)
        for k in range(3):
            ctx.load_tracks(k, pop[k]["tracks"], pop[k]["slots"] if scheme == "sparse" else None)
        g = ctx.step()
        compare_counts(g, r, what="%s/%s" % (layout, scheme))
        assert int(g["secondaries"][2]) == forced[0] + forced[1] and int(g["secondaries"][0]) == forced[2]
        for k in range(3):
            compare_tracks(ctx.read_tracks(k), o.read_tracks(k, pop[0]["tracks"].dtype), "%s/%s" % (layout, scheme))
        ctx.destroy()


# ------------------------------------------------------------------------ edge cases ---------
def test_edge_cases_empty_overflow_invalid_reset():
    from paper_2302_08252_b200 import AdeptError
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    ctx = _ctx(geo, tab, layout="soa", scheme="dense", capacity=128, seed=1)
    c = ctx.step()                                   # empty step: nothing happens, not counted
    assert c["live"].sum() == 0 and c["iterations"] == 0 and c["steps"].sum() == 0
    r = ctx.run()
    assert r["iterations"] == 0 and r["edep_slab"].sum() == 0
    bad = gen_primaries(1, 10.0)
    bad["ekin"] = 1e6                                # above e_max
    with pytest.raises(AdeptError) as e:
        ctx.inject(bad)
    assert e.value.code == -1
    bad = gen_primaries(1, 10.0)
    bad["pos"][0, 0] = 1e3                           # outside the transverse box
    with pytest.raises(AdeptError):
        ctx.inject(bad)
    # overflow: 128 x 10 MeV showers need more than 128 slots per kind
    ctx.inject(gen_primaries(128, 10.0))
    with pytest.raises(AdeptError) as e:
        ctx.run()
    assert e.value.code == -2
    with pytest.raises(AdeptError) as e:
        ctx.step()
    assert e.value.code == -4
    ctx.reset()
    ctx.inject(gen_primaries(2, 10.0))
    o = Oracle(geo, tab, seed=1)
    o.inject(gen_primaries(2, 10.0))
    o.run()
    compare_counts(ctx.run(), o.result())
    ctx.destroy()
    with pytest.raises(AdeptError):
        _ctx(geo, tab, layout="soa", scheme="dense", capacity=0)


# ------------------------------------------------------------- event sharding ---
def test_sliced_runs_add_up_to_the_unsliced_run():
    """adept_set_primary_index: two contexts that each take a slice of the primary list (what two
    ranks of a multi-GPU run do, here one after the other on one device) add up to the single run."""
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    prim = gen_primaries(13, 10.0)
    o = Oracle(geo, tab, seed=21)
    o.inject(prim)
    o.run()
    r = o.result()
    parts = []
    for lo, hi in ((0, 7), (7, 13)):
        ctx = _ctx(geo, tab, layout="aosoa32", scheme="dense", capacity=4096, seed=21)
        ctx.set_primary_index(lo)
        ctx.inject(prim[lo:hi])
        parts.append(ctx.run())
        ctx.destroy()
    for k in ("steps", "secondaries", "killed", "escaped_n"):
        assert (parts[0][k] + parts[1][k] == r[k]).all(), k
    assert max(p["iterations"] for p in parts) == r["iterations"]
    assert np.allclose(parts[0]["edep_layer"] + parts[1]["edep_layer"], r["edep_layer"], rtol=1e-9, atol=1e-12)


# ----------------------------------------------------- instrumented build ---
@pytest.mark.parametrize("layout", LAYOUTS)
def test_instrumented_dense_counts_follow_the_access_rules(layout):
    """PAPER.md:115/123 per-field counts, PAPER.md:131/135 per-row heatmap, PAPER.md:137 per-slot use.
    Dense double buffer: a step reads all 14 words of every live track once and writes all 14 words
    of every track that enters the next arrays (survivor or secondary)."""
    c = CONFIGS["single_step"]
    geo, tab = geometry_for("single_step"), tables_for("single_step")
    pop = gen_tracks(6000 + 13, c["seed"], geo, c["e_max"], c["fractions"])
    for k in range(3):
        pop[k]["nial"][::5] = 1e-30                    # plenty of interactions and secondaries
    cap = 8192
    ctx = _ctx(geo, tab, layout=layout, scheme="dense", capacity=cap, seed=3, instrument=True)
    n_in = [p.shape[0] for p in pop]
    for k in range(3):
        ctx.load_tracks(k, pop[k])
    counts = ctx.step()
    cnt = ctx.read_counters()
    rw, lines, slots = cnt["field_rw"], cnt["lines"], cnt["slots"]
    assert counts["secondaries"].sum() > 100
    for k in range(3):
        assert (rw[k, :, 0] == n_in[k]).all()
        assert (rw[k, :, 1] == counts["live"][k]).all()
        assert int(lines[k].sum()) == int(rw[k].sum()) == int(slots[k].sum())
        cur, nxt = slots[k][:cap], slots[k][cap:]       # parity 0 is current before the step
        assert (cur[:n_in[k]] == 14).all() and (cur[n_in[k]:] == 0).all()
        assert (nxt[:counts["live"][k]] == 14).all() and (nxt[counts["live"][k]:] == 0).all()
        # heatmap rows: every 128-byte line of the used part of the current buffer was touched
        from paper_2302_08252_b200 import LAYOUTS as LAY, field_offset
        touched = {field_offset(LAY[layout], cap, s, f, kind=k) // 128 for s in (0, n_in[k] - 1) for f in range(14)}
        assert all(lines[k][t] > 0 for t in touched)
    ctx.destroy()


def test_instrumented_sparse_writes_only_what_changed():
    """Sparse single buffer: 14 reads per step; in-place write-back of changed words only -- ids are
    written for new tracks only, and no field is written more often than twice per live track
    (once by each half of the step) plus once per secondary."""
    c = CONFIGS["single_step"]
    geo, tab = geometry_for("single_step"), tables_for("single_step")
    pop = gen_tracks(5000, c["seed"], geo, c["e_max"], c["fractions"])
    for k in range(3):
        pop[k]["nial"][::4] = 1e-30
    ctx = _ctx(geo, tab, layout="soa", scheme="sparse", capacity=16384, seed=3, instrument=True)
    n_in = [p.shape[0] for p in pop]
    for k in range(3):
        ctx.load_tracks(k, pop[k])
    counts = ctx.step()
    rw = ctx.read_counters()["field_rw"]
    ID_LO, ID_HI, STEP, EKIN = 11, 12, 13, 6
    for k in range(3):
        assert (rw[k, :, 0] == n_in[k]).all()
        born = int(counts["secondaries"][k])
        assert rw[k, ID_LO, 1] == born and rw[k, ID_HI, 1] == born
        survivors = int(counts["live"][k]) - born
        assert rw[k, STEP, 1] >= survivors + born          # every survivor's step counter changed
        assert (rw[k, :, 1] <= 2 * n_in[k] + born).all()
    assert rw[2, EKIN, 1] < rw[2, STEP, 1]                  # photons rarely change energy
    assert rw[0, EKIN, 1] >= int(counts["live"][0]) - int(counts["secondaries"][0])   # electrons always do
    ctx.destroy()


# ------------------------------------------- BASELINE.json sizes, bench.py's launch configuration ---
_FULL_SIZE_CACHE = {}


def _full_size_reference(n):
    """Population and oracle step of config 3 at n tracks (computed once per size)."""
    if n not in _FULL_SIZE_CACHE:
        _FULL_SIZE_CACHE.clear()                       # one size at a time: the arrays are ~1 GB each
        c = CONFIGS["single_step"]
        geo, tab = geometry_for("single_step"), tables_for("single_step")
        pop = gen_tracks(n, c["seed"], geo, c["e_max"], c["fractions"])
        o = Oracle(geo, tab, seed=c["seed"])
        for k in range(3):
            o.load_tracks(k, pop[k])
        o.step()
        ref = [sort_by_id(o.read_tracks(k, pop[0].dtype)) for k in range(3)]
        _FULL_SIZE_CACHE[n] = (geo, tab, pop, o.result(), ref)
        o.close()
    return _FULL_SIZE_CACHE[n]


@pytest.mark.parametrize("layout,scheme,n", [("aosoa32", "dense", 1 << 24),
                                             ("soa", "dense", 1 << 23), ("soa16", "dense", 1 << 23),
                                             ("aos", "dense", 1 << 23), ("aosoa64", "dense", 1 << 23),
                                             ("aos", "sparse", 1 << 23), ("soa", "sparse", 1 << 23),
                                             ("aosoa32", "sparse", 1 << 23), ("hc16", "dense", 1 << 23),
                                             ("hc16", "sparse", 1 << 23)])
def test_single_step_at_full_size_counts_and_every_track(layout, scheme, n):
    """Config 3 as bench.py times it: 2^24 tracks, dense double buffer, AoSoA-32, one adept_step --
    and 2^23 tracks in seven more layout x scheme variants; all above the population at which the
    library switches to its 1024-thread CTAs.  All integer counts and the per-slab deposits against
    the oracle's full-size step, and EVERY surviving / created track compared word for word (sorted
    by id), so that every lane position of the 1024-thread shape is covered."""
    c = CONFIGS["single_step"]
    geo, tab, pop, r, ref = _full_size_reference(n)
    cap = int(max(p.shape[0] for p in pop) * 1.25) + 4096
    if scheme == "sparse":
        cap = int(max(p.shape[0] for p in pop) * 1.6) + 4096      # slots of new tracks come on top of the old
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=cap, seed=c["seed"])
    for k in range(3):
        ctx.load_tracks(k, pop[k])
    counts = ctx.step()
    compare_counts(counts, r, what="full size")
    g = ctx.result()
    assert np.allclose(g["edep_slab"], r["edep_slab"], rtol=1e-9, atol=1e-6)
    assert abs(g["e_escaped"] - r["e_escaped"]) <= 1e-9 * r["e_escaped"]
    if scheme == "sparse":       # rule S30: bump allocation on top of the loaded population
        assert (g["slots_used"] == np.array([p.shape[0] for p in pop], dtype=np.uint64) + r["secondaries"]).all()
    for k in range(3):
        a = sort_by_id(ctx.read_tracks(k))
        assert a.shape[0] == ref[k].shape[0] == int(counts["live"][k])
        same = a.view(np.uint8).reshape(-1, 56) == ref[k].view(np.uint8).reshape(-1, 56)
        assert same.all(), "kind %d: %d tracks differ" % (k, int((~same.all(axis=1)).sum()))
    ctx.destroy()


# ------------------------------------------------------------------ ragged and empty inputs ---
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("layout", LAYOUTS)
def test_ragged_tile_sizes_and_empty_kinds(layout, scheme):
    """Populations around the tile (128) and warp (32) boundaries, kinds with no track at all, every
    track forced to interact (the parked queue runs full): two steps each, compared per track."""
    c = CONFIGS["single_step"]
    geo, tab = geometry_for("single_step"), tables_for("single_step")
    rng = np.random.default_rng(77)
    cases = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (31, 33, 32), (127, 129, 128), (255, 0, 257), (0, 385, 1), (640, 3, 1000)]
    for ci, sizes in enumerate(cases):
        n = sum(sizes)
        fr = tuple(s / n for s in sizes)
        pop = gen_tracks(n, 100 + ci, geo, c["e_max"], fr)
        assert tuple(p.shape[0] for p in pop) == sizes, (sizes, [p.shape[0] for p in pop])
        for k in range(3):
            if ci % 2 == 1 and pop[k].shape[0]:
                pop[k]["nial"][:, :] = np.float32(1e-30)          # every track interacts this step
            if k == 1 and pop[k].shape[0]:
                pop[k]["ekin"][rng.random(pop[k].shape[0]) < 0.3] = np.float32(0.05)   # e+ at rest
        o = Oracle(geo, tab, seed=5)
        ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=4096, seed=5)
        for k in range(3):
            if pop[k].shape[0]:
                o.load_tracks(k, pop[k])
                ctx.load_tracks(k, pop[k])
        for it in range(2):
            o.step()
            counts = ctx.step()
            compare_counts(counts, o.result(), what="%s/%s case %d step %d" % (layout, scheme, ci, it))
            for k in range(3):
                assert compare_tracks(ctx.read_tracks(k), o.read_tracks(k, pop[0].dtype), "case %d kind %d" % (ci, k)) == 0
        g, r = ctx.result(), o.result()
        assert np.allclose(g["edep_slab"], r["edep_slab"], rtol=1e-9, atol=1e-7)
        ctx.destroy()


def test_tallies_are_bit_identical_across_layouts_schemes_and_runs():
    """DESIGN.md reading 33: energies are accumulated in 64-bit fixed point, so the sums do not
    depend on the order in which threads, warps and CTAs arrive -- nor on layout or scheme."""
    c = CONFIGS["full"]
    geo, tab = geometry_for("full"), tables_for("full")
    prim = gen_primaries(40, c["e_primary"])
    ref = None
    for layout, scheme in (("aosoa32", "dense"), ("aosoa32", "dense"), ("soa", "sparse"), ("aos", "dense"), ("soa16", "sparse")):
        ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=1 << 18, seed=c["seed"])
        ctx.inject(prim)
        g = ctx.run()
        ctx.destroy()
        bits = (g["edep_slab"].tobytes(), np.float64(g["e_escaped"]).tobytes())
        if ref is None:
            ref = bits
        assert bits == ref, (layout, scheme)


# ---------------------------------------------- rule R4 / locator / S31 / S24 on the device ---
def _gun(kinds, zs, ekin=5.0):
    from workloads import PRIMARY_DTYPE
    p = np.zeros(len(zs), dtype=PRIMARY_DTYPE)
    p["kind"] = kinds
    p["pos"][:, 2] = np.asarray(zs, dtype=np.float32)
    p["dir"][:, 2] = 1.0
    p["ekin"] = np.float32(ekin)
    return p


@pytest.mark.parametrize("scheme", SCHEMES)
def test_inject_mixed_kinds_ids_and_slabs(scheme):
    """adept_inject: rule R4 ids (against the numpy Philox of tests/helpers.py and the oracle) for
    p = 0, 1, 2^32 + 3 under two seeds, and the slab locator at z = 0, inside an absorber, exactly on
    abs_mm, inside a gap, on a layer boundary and on the last plane, for a mixed e-/e+/gamma array."""
    from tests.helpers import primary_ids_np
    from workloads import Geometry
    geo = Geometry(n_layers=3, abs_mm=2.5, gap_mm=5.5, half_xy_mm=50.0)       # pitch 8, exact in binary
    tab = tables_for("tiny")
    zs = [0.0, 1.0, 2.5, 5.0, 8.0, 10.5, 15.999, 16.0, 18.5, 24.0]
    want_vol = np.array([0, 0, 1, 1, 2, 3, 3, 4, 5, 5])
    kinds = np.array([2, 0, 1, 0, 2, 1, 0, 0, 2, 1])
    prim = _gun(kinds, zs)
    for seed in (0x1234, 0xABCDEF0123456789):
        for first in (0, 1, (1 << 32) + 3):
            ctx = _ctx(geo, tab, layout="aosoa32", scheme=scheme, capacity=256, seed=seed)
            o = Oracle(geo, tab, seed=seed)
            ctx.set_primary_index(first)
            o.set_primary_index(first)
            ctx.inject(prim)
            o.inject(prim)
            lo, hi = primary_ids_np(first + np.arange(len(zs), dtype=np.uint64), seed)
            for k in range(3):
                g = ctx.read_tracks(k)
                sel = kinds == k
                assert compare_tracks(g, o.read_tracks(k, g.dtype), "inject kind %d" % k) == 0
                order = np.argsort(hi[sel].astype(np.uint64) << np.uint64(32) | lo[sel].astype(np.uint64))
                gs = sort_by_id(g)
                assert (gs["id_lo"] == lo[sel][order]).all() and (gs["id_hi"] == hi[sel][order]).all()
                assert (gs["vol"] == want_vol[sel][order]).all()
                assert (gs["step"] == 0).all() and (gs["nial"] == -1.0).all()
            assert abs(ctx.result()["e_injected"] - o.result()["e_injected"]) < 1e-9
            ctx.destroy()


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("layout", ("aos", "soa", "aosoa32"))
def test_runaway_guard_and_continuous_loss_cases(layout, scheme):
    """The oracle's S31 and S24 pins (tests/test_oracle_transport.py) through adept_load_tracks +
    adept_step: tracks at step 2^20 - 2 / 2^20 - 1 of every kind (killed, energy into the post-step
    slab); the midpoint rule on a two-node table; a step that reaches the range (E_post = 0)."""
    from workloads import Geometry
    from workloads.tables import GROUP_ELEC, Q_STOP, MC2, constant_tables
    geo = Geometry(n_layers=2, abs_mm=2.5, gap_mm=5.5, half_xy_mm=50.0)
    tab = constant_tables(16, 0.1, 100.0, 0.1)
    e0 = np.float32(3.25)
    for kind in range(3):
        for step0, dies in (((1 << 20) - 2, False), ((1 << 20) - 1, True)):
            t = make_tracks(130, ekin=e0, step=step0)
            ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=512, seed=0)
            o = Oracle(geo, tab, seed=0)
            ctx.load_tracks(kind, t)
            o.load_tracks(kind, t)
            counts = ctx.step()
            o.step()
            compare_counts(counts, o.result(), what="S31 kind %d step0 %d" % (kind, step0))
            assert compare_tracks(ctx.read_tracks(kind), o.read_tracks(kind, t.dtype)) == 0
            g = ctx.result()
            if dies:
                rest = float(np.float32(2.0) * np.float32(MC2)) if kind == 1 else 0.0
                assert int(counts["live"][kind]) == 0 and int(counts["killed"][kind]) == 130
                assert abs(g["edep_slab"][1] - 130 * (float(e0) + rest)) < 1e-6 and g["edep_slab"][[0, 2, 3]].sum() == 0
            else:
                assert int(counts["live"][kind]) == 130 and g["edep_slab"].sum() == 0
            ctx.destroy()
    # S24 on a two-node table with S linear in ln E (closed form in the oracle's pin) and the stop rule
    geo = Geometry(n_layers=1, abs_mm=1e3, gap_mm=1.0, half_xy_mm=1e6)
    for rng_mm, s_lo, s_hi in ((50.0, 0.5, 1.5), (0.05, 1e-3, 1e-3), (0.3, 1e-3, 1e-3)):
        tab = constant_tables(1, 0.1, 100.0, 0.1, brems=0.0, rng=rng_mm)
        tab.data[:, GROUP_ELEC, Q_STOP, 0] = s_lo
        tab.data[:, GROUP_ELEC, Q_STOP, 1] = s_hi
        E = np.float32([90.0, 50.0, 20.0, 13.0, 2.0, 7.5])
        for kind in (0, 1):
            t = make_tracks(E.shape[0], ekin=E, pos=(0, 0, 500.0))
            ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=128, seed=0)
            o = Oracle(geo, tab, seed=0)
            ctx.load_tracks(kind, t)
            o.load_tracks(kind, t)
            for it in range(2):        # second step: the stopped e+ (ekin = 0) annihilate (rule S17)
                counts = ctx.step()
                o.step()
                compare_counts(counts, o.result(), what="S24 range %g kind %d" % (rng_mm, kind))
                for k in range(3):
                    assert compare_tracks(ctx.read_tracks(k), o.read_tracks(k, t.dtype)) == 0
            assert np.allclose(ctx.result()["edep_slab"], o.result()["edep_slab"], rtol=1e-9, atol=1e-9)
            ctx.destroy()


def test_device_math_exhaustive_bit_equality():
    """lg / ex / sincos2pi evaluated on the device for EVERY fp32 of the
    used domains ([1e-8, 1e5]; +-[1e-6, 20]; the whole 2^23-point u grid) equal the oracle's bit for
    bit; u01 over the whole grid."""
    import torch
    from paper_2302_08252_b200 import dev_math

    def every_float(lo, hi, chunk=1 << 25):
        a, b = int(np.float32(lo).view(np.uint32)), int(np.float32(hi).view(np.uint32))
        for first in range(a, b, chunk):
            yield np.arange(first, min(first + chunk, b), dtype=np.uint32).view(np.float32)

    n = 0
    for x in every_float(1e-8, 1e5):
        y = dev_math(2, torch.from_numpy(x).cuda(), torch.float32, (x.shape[0],)).cpu().numpy()
        assert (y.view(np.uint32) == math_fns.lg(x).view(np.uint32)).all()
        n += x.shape[0]
    for sign in (1.0, -1.0):
        for x in every_float(1e-6, 20.0):
            x = np.float32(sign) * x
            y = dev_math(3, torch.from_numpy(x).cuda(), torch.float32, (x.shape[0],)).cpu().numpy()
            assert (y.view(np.uint32) == math_fns.ex(x).view(np.uint32)).all()
            n += x.shape[0]
    assert n > 7.5e8
    xs = (np.arange(1 << 23, dtype=np.uint64) << np.uint64(9)).astype(np.uint32)
    u = dev_math(1, torch.from_numpy(xs.view(np.int32)).cuda(), torch.float32, (xs.shape[0],)).cpu().numpy()
    assert (u.view(np.uint32) == math_fns.u01(xs).view(np.uint32)).all()
    sc = dev_math(4, torch.from_numpy(u).cuda(), torch.float32, (u.shape[0], 2)).cpu().numpy()
    s, c = math_fns.sincos2pi(u)
    assert (sc[:, 0].view(np.uint32) == s.view(np.uint32)).all() and (sc[:, 1].view(np.uint32) == c.view(np.uint32)).all()
    y = dev_math(2, torch.from_numpy(u).cuda(), torch.float32, (u.shape[0],)).cpu().numpy()
    assert (y.view(np.uint32) == math_fns.lg(u).view(np.uint32)).all()


# ------------------------------------------------------------- host-side contract ---
def test_two_live_contexts_with_different_tables_step_alternately():
    """The dynamic shared-memory limit of a kernel instantiation is shared by all contexts of the
    process: a later context with smaller tables must not lower it under an earlier, larger one."""
    big_geo, big_tab = geometry_for("full"), tables_for("full")          # 257 nodes, 100 slabs
    small_geo, small_tab = geometry_for("tiny"), tables_for("tiny")      # 65 nodes, 8 slabs
    a = _ctx(big_geo, big_tab, layout="aosoa32", scheme="dense", capacity=1 << 16, seed=2)
    b = _ctx(small_geo, small_tab, layout="aosoa32", scheme="dense", capacity=4096, seed=1)
    a.inject(gen_primaries(3, 1000.0))
    b.inject(gen_primaries(16, 10.0))
    oa, ob = Oracle(big_geo, big_tab, seed=2), Oracle(small_geo, small_tab, seed=1)
    oa.inject(gen_primaries(3, 1000.0))
    ob.inject(gen_primaries(16, 10.0))
    for it in range(30):
        ca, cb = a.step(), b.step()
        oa.step()
        ob.step()
        compare_counts(ca, oa.result(), what="big context, iteration %d" % it)
        compare_counts(cb, ob.result(), what="small context, iteration %d" % it)
    oa.run()
    ob.run()
    compare_counts(a.run(), oa.result())
    compare_counts(b.run(), ob.result())
    a.destroy()
    b.destroy()


def test_load_tracks_rejects_bad_records_and_slots():
    from paper_2302_08252_b200 import AdeptError
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    good = make_tracks(300, ekin=1.0)
    for scheme in SCHEMES:
        ctx = _ctx(geo, tab, layout="soa", scheme=scheme, capacity=1024, seed=1)
        for field, value in (("vol", 2 * geo.n_layers), ("step", 1 << 20), ("ekin", 0.01), ("ekin", 1e5),
                             ("ekin", np.nan), ("dir", (0.0, 0.0, 0.0)), ("dir", (np.inf, 0.0, 1.0)),
                             ("pos", (np.nan, 0.0, 0.0)), ("nial", (np.nan, 1.0, 1.0))):
            bad = good.copy()
            bad[field][257] = value
            with pytest.raises(AdeptError) as e:
                ctx.load_tracks(0, bad)
            assert e.value.code == -1, (field, value)
            assert ctx.step()["live"].sum() == 0                     # nothing was changed
        low = good.copy()
        low["ekin"][::3] = 0.01                                      # allowed for e+ only (rule S17)
        ctx.load_tracks(1, low)
        assert int(ctx.step()["steps"][1]) == 300
        ctx.destroy()
    ctx = _ctx(geo, tab, layout="aos", scheme="sparse", capacity=1024, seed=1)
    slots = np.arange(300, dtype=np.uint32) * 3
    dup = slots.copy()
    dup[200] = dup[17]
    for bad_slots in (dup, slots + 200):                             # duplicate; beyond the capacity
        with pytest.raises(AdeptError) as e:
            ctx.load_tracks(0, good, bad_slots)
        assert e.value.code == -1
    ctx.load_tracks(0, good, slots)
    with pytest.raises(AdeptError):                                  # slot 5 lies below the allocator's top: not free
        ctx.load_tracks(0, good[:1], np.array([5], dtype=np.uint32))
    ctx.load_tracks(0, good[:2], np.array([1000, 950], dtype=np.uint32))
    o = Oracle(geo, tab, seed=1)
    o.load_tracks(0, np.concatenate([good, good[:2]]))
    o.step()
    compare_counts(ctx.step(), o.result())
    ctx.destroy()


def test_run_counts_real_iterations_against_the_limit():
    """adept_run(max_iterations): progress is what the device counted (iterations with something
    alive), the limit is tested before the next batch is injected, and a run can be resumed."""
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    prim = gen_primaries(6, 10.0)
    o = Oracle(geo, tab, seed=9)
    o.queue(prim)
    o.run_batched(2)
    r = o.result()
    ctx = _ctx(geo, tab, layout="soa", scheme="dense", capacity=4096, seed=9, batch_primaries=2)
    ctx.inject(prim)
    done = 0
    while True:
        g = ctx.run(7)
        assert g["iterations"] - done <= 7
        if g["iterations"] == done:
            break
        assert g["iterations"] - done == 7 or g["live"].sum() == 0
        done = g["iterations"]
    compare_counts(g, r)
    assert g["iterations"] == r["iterations"]
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-12)
    ctx.destroy()


# ----------------------------------------------------------- slot recycling --
@pytest.mark.parametrize("layout", ("aos", "soa", "aosoa32", "soa16", "hc16"))
def test_sparse_slot_recycling_keeps_results_and_bounds_the_footprint(layout):
    """ADEPT_FLAG_RECYCLE_SLOTS (include/adept.h): the slot of every track that ends goes onto a ring
    and secondaries take recycled slots first.  Slots carry no physics, so every count, every tally and
    every surviving track must equal the oracle's -- iteration by iteration on the tiny shower, and
    over 100 x 1 GeV showers in a buffer far smaller than the never-recycle policy needs (PAPER.md:137:
    2044 against 45509 slots)."""
    RECYCLE = 1
    c = CONFIGS["tiny"]
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    prim = gen_primaries(c["n_primaries"], c["e_primary"])
    o = Oracle(geo, tab, seed=c["seed"])
    o.inject(prim)
    ctx = _ctx(geo, tab, layout=layout, scheme="sparse", capacity=c["capacity"], seed=c["seed"], flags=RECYCLE)
    ctx.inject(prim)
    it = 0
    while sum(o.live(k) for k in range(3)):
        o.step()
        compare_counts(ctx.step(), o.result(), what="iteration %d" % it)
        for k in range(3):
            compare_tracks(ctx.read_tracks(k), o.read_tracks(k, make_tracks(1).dtype), "iteration %d kind %d" % (it, k))
        it += 1
    r, g = o.result(), ctx.result()
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-12)
    never = np.array([c["n_primaries"], 0, 0], dtype=np.uint64) + r["secondaries"]
    assert (g["slots_used"] <= never).all() and g["slots_used"].sum() < never.sum()
    ctx.destroy()

    c = CONFIGS["full"]
    geo, tab = geometry_for("full"), tables_for("full")
    prim = gen_primaries(100, c["e_primary"])
    o = Oracle(geo, tab, seed=c["seed"])
    o.inject(prim)
    o.run()
    r = o.result()
    cap = 1 << 14                                   # peak live per kind is ~6e3; e- created in total ~5.8e4
    assert r["secondaries"][0] > 3 * cap
    ctx = _ctx(geo, tab, layout=layout, scheme="sparse", capacity=cap, seed=c["seed"], flags=RECYCLE)
    ctx.inject(prim)
    g = ctx.run()
    compare_counts(g, r)
    assert g["iterations"] == r["iterations"] and g["overflow"] == 0
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-9)
    assert (g["slots_used"] <= cap).all()
    ctx.destroy()
    # the paper's policy in the same buffer: it overflows, and says so
    from paper_2302_08252_b200 import AdeptError
    ctx = _ctx(geo, tab, layout=layout, scheme="sparse", capacity=cap, seed=c["seed"])
    ctx.inject(prim)
    with pytest.raises(AdeptError) as e:
        ctx.run()
    assert e.value.code == -2
    ctx.destroy()


def test_recycling_flag_is_validated_and_ignored_by_the_dense_scheme():
    from paper_2302_08252_b200 import AdeptError
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    with pytest.raises(AdeptError):
        _ctx(geo, tab, layout="soa", scheme="sparse", capacity=4096, flags=2)
    prim = gen_primaries(16, 10.0)
    a = _ctx(geo, tab, layout="soa", scheme="dense", capacity=4096, seed=1, flags=1)
    b = _ctx(geo, tab, layout="soa", scheme="dense", capacity=4096, seed=1)
    a.inject(prim); b.inject(prim)
    ra, rb = a.run(), b.run()
    compare_counts(ra, rb)
    assert (ra["edep_slab"] == rb["edep_slab"]).all() and (ra["slots_used"] == rb["slots_used"]).all()
    a.destroy(); b.destroy()


# ------------------------------------------------------------------ config 5 at full size ----------
@pytest.mark.slow
@pytest.mark.parametrize("layout,scheme,flags", [("aosoa32", "dense", 0), ("aos", "sparse", 1)])
def test_heavy_showers_at_full_size_match_the_oracle(layout, scheme, flags):
    """BASELINE.json configs[4]: 10 000 x 10 GeV e-, 8 Mi slots per kind, run to completion -- every
    count bit-exact, per-layer deposits within 1e-4 (the oracle needs ~80 s on one host core).  The
    sparse single buffer holds the run in the same 8 Mi slots only with slot recycling (the e- created
    in total are ~5.7e7, SURVEY.md:583)."""
    c = CONFIGS["heavy"]
    geo, tab = geometry_for("heavy"), tables_for("heavy")
    prim = gen_primaries(c["n_primaries"], c["e_primary"])
    r = _heavy_reference()
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=c["capacity"], seed=c["seed"], flags=flags)
    ctx.inject(prim)
    g = ctx.run()
    compare_counts(g, r)
    assert g["iterations"] == r["iterations"] and g["overflow"] == 0
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-9)
    assert abs(g["e_escaped"] - r["e_escaped"]) <= 1e-9 * r["e_injected"]
    assert abs(g["edep_slab"].sum() + g["e_escaped"] - g["e_injected"]) < 1e-6 * g["e_injected"]
    if scheme == "sparse":
        assert (g["slots_used"] <= c["capacity"]).all() and r["secondaries"][0] > 4 * c["capacity"]
    ctx.destroy()


_HEAVY = {}


def _heavy_reference():
    if not _HEAVY:
        c = CONFIGS["heavy"]
        o = Oracle(geometry_for("heavy"), tables_for("heavy"), seed=c["seed"])
        o.inject(gen_primaries(c["n_primaries"], c["e_primary"]))
        o.run()
        _HEAVY.update(o.result())
        o.close()
    return _HEAVY


# ------------------------------------------------- extended physics ----------
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("layout", ("aos", "soa", "aosoa32", "soa16", "hc16"))
def test_extended_physics_matches_oracle(layout, scheme):
    """adept_tables.physics = 1 (rules X36 delta rays on nial[1], X37 Klein-Nishina rejection sampling):
    the tiny shower track by track in every iteration, then 100 x 1 GeV showers to completion."""
    c = CONFIGS["tiny"]
    geo, tab = geometry_for("tiny"), tables_for("tiny", physics=1)
    prim = gen_primaries(c["n_primaries"], c["e_primary"])
    o = Oracle(geo, tab, seed=c["seed"])
    o.inject(prim)
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=c["capacity"], seed=c["seed"])
    ctx.inject(prim)
    it = 0
    while sum(o.live(k) for k in range(3)):
        o.step()
        compare_counts(ctx.step(), o.result(), what="iteration %d" % it)
        for k in range(3):
            compare_tracks(ctx.read_tracks(k), o.read_tracks(k, make_tracks(1).dtype), "iteration %d kind %d" % (it, k))
        it += 1
    r, g = o.result(), ctx.result()
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-12)
    ctx.destroy()
    basic = Oracle(geo, tables_for("tiny"), seed=c["seed"])
    basic.inject(prim)
    basic.run()
    assert r["secondaries"][0] > basic.result()["secondaries"][0]        # the delta rays are there

    c = CONFIGS["full"]
    geo, tab = geometry_for("full"), tables_for("full", physics=1)
    prim = gen_primaries(100, c["e_primary"])
    o = Oracle(geo, tab, seed=c["seed"])
    o.inject(prim)
    o.run()
    r = o.result()
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=1 << 19, seed=c["seed"])
    ctx.inject(prim)
    g = ctx.run()
    compare_counts(g, r)
    assert g["iterations"] == r["iterations"]
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-9)
    assert abs(g["edep_slab"].sum() + g["e_escaped"] - g["e_injected"]) < 1e-6 * g["e_injected"]
    ctx.destroy()


def test_extended_physics_single_step_population_and_validation():
    """One step of a config-3-like population under the extended rules, every track compared; the
    variant is refused where it is not built (instrumented contexts, slot recycling)."""
    from paper_2302_08252_b200 import AdeptError
    geo, tab = geometry_for("single_step"), tables_for("single_step", physics=1)
    pop = gen_tracks(300_001, 11, geo, CONFIGS["single_step"]["e_max"])
    for p in pop:                                   # spent interaction lengths: everything re-samples
        p["nial"][::3] = -1.0
    o = Oracle(geo, tab, seed=3)
    for k in range(3):
        o.load_tracks(k, pop[k])
    o.step()
    r = o.result()
    for layout, scheme in (("aosoa32", "dense"), ("soa", "dense"), ("aos", "sparse"), ("soa", "sparse")):
        ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=1 << 19, seed=3)
        for k in range(3):
            ctx.load_tracks(k, pop[k])
        compare_counts(ctx.step(), r, what=layout + scheme)
        for k in range(3):
            assert compare_tracks(ctx.read_tracks(k), o.read_tracks(k, pop[k].dtype), "%s %s kind %d" % (layout, scheme, k)) == 0
        ctx.destroy()
    with pytest.raises(AdeptError):
        _ctx(geo, tab, layout="soa", scheme="dense", capacity=4096, instrument=True)
    with pytest.raises(AdeptError):
        _ctx(geo, tab, layout="soa", scheme="sparse", capacity=4096, flags=1)


# ------------------------------------------------------------------ timing variant -----------------
def test_timing_variant_computes_the_same_and_fills_its_section_clocks():
    """libadept_b200_timing.so (-DADEPT_TIMING_SECTIONS, include/adept.h): same results as the plain
    library, and the per-section warp-cycle sums bench.py's sweep reads are there."""
    from paper_2302_08252_b200 import lib
    assert lib().adept_timing_sections() == 0 and lib("timing").adept_timing_sections() == 1
    pop = gen_sweep(0.3, span=1 << 16)
    geo, tab = geometry_for("sweep"), tables_for("sweep")
    for scheme in SCHEMES:
        res = []
        for variant in (None, "timing"):
            ctx = _ctx(geo, tab, layout="aosoa32", scheme=scheme, capacity=1 << 17, seed=4, variant=variant)
            for k in range(3):
                ctx.load_tracks(k, pop[k]["tracks"], pop[k]["slots"] if scheme == "sparse" else None)
            counts = ctx.step()
            sec = ctx.read_sections()
            res.append((counts, ctx.result(), [sort_by_id(ctx.read_tracks(k)) for k in range(3)], sec))
            ctx.destroy()
        compare_counts(res[0][0], res[1][0])
        assert (res[0][1]["edep_slab"] == res[1][1]["edep_slab"]).all()
        for a, b in zip(res[0][2], res[1][2]):
            assert (a.view(np.uint8) == b.view(np.uint8)).all()
        assert res[0][3].sum() == 0                                   # the plain library keeps no clocks
        s = res[1][3]
        assert (s[1:6] > 0).all() and s[4] + s[5] < s[:6].sum()       # load, move, interact, alloc, store all ran
        assert s[6] > 0                                               # launch timeline (ns)


@pytest.mark.parametrize("scheme", SCHEMES)
def test_extended_physics_forced_interactions(scheme):
    """Every track's step ends in the process under test: delta rays of e- and e+ (X36), annihilation
    in flight (X38), Klein-Nishina Compton (X37) -- counts and all track words against the oracle."""
    from workloads.tables import constant_tables
    from workloads import Geometry
    geo = Geometry(n_layers=2, abs_mm=50.0, gap_mm=50.0, half_xy_mm=1e4)
    tab = constant_tables(16, 0.1, 100.0, 0.1, physics=1, delta=1.0, annih=1.0, compt=1.0, stop=0.0)
    n = 5000 + 77
    rng = np.random.default_rng(12)
    cases = ((0, (1e6, 1e-30, 1e6)), (1, (1e6, 1e-30, 1e6)), (1, (1e6, 1e6, 1e-30)), (2, (1e6, 1e-30, 1e6)))
    for layout in ("aosoa32", "aos", "hc16"):
        for kind, nial in cases:
            t = make_tracks(n, pos=(0, 0, 25.0), ekin=1.0, nial=nial, id0=1 + 100000 * kind)
            # from 0.12 MeV: below 2 e_cut = 0.2 MeV the delta-ray interval is empty (guard of rule X36)
            t["ekin"] = np.exp(rng.uniform(np.log(0.12), np.log(90.0), n)).astype(np.float32)
            ct = rng.uniform(-1, 1, n)
            ph = rng.uniform(0, 2 * np.pi, n)
            d = np.stack([np.sqrt(1 - ct * ct) * np.cos(ph), np.sqrt(1 - ct * ct) * np.sin(ph), ct], 1)
            t["dir"] = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
            o = Oracle(geo, tab, seed=0)
            o.load_tracks(kind, t)
            o.step()
            r = o.result()
            assert r["secondaries"].sum() >= n // 2
            ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=1 << 14, seed=0)
            ctx.load_tracks(kind, t)
            compare_counts(ctx.step(), r, what="%s kind %d %s" % (layout, kind, nial))
            for k in range(3):
                assert compare_tracks(ctx.read_tracks(k), o.read_tracks(k, t.dtype), "kind %d" % k) == 0
            g = ctx.result()
            assert np.allclose(g["edep_slab"], r["edep_slab"], rtol=1e-9, atol=1e-9)
            # the library's own state is a valid input: no e- or photon below the cut comes out of a step, so
            # what adept_read_tracks returns adept_load_tracks accepts (it refuses such records with EINVAL)
            back = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=1 << 14, seed=0)
            for k in range(3):
                live = ctx.read_tracks(k)
                if k != 1:
                    assert (live["ekin"] >= np.float32(0.1)).all()
                if live.shape[0]:
                    back.load_tracks(k, live)
            back.destroy()
            ctx.destroy()


# ------------------------------------------------------------------ iteration control --------------
def test_snapshot_rewind_and_launch_index_wrap():
    """include/adept.h "Workspace": a workspace copy + launch index rewinds a context; and the launch
    index, by which the device keeps its per-iteration counters three deep, wraps at a multiple of 6
    just below 2^32 without a seam (the context is started a few launches before the wrap by setting
    the index and the control block's `closed` word, byte 248, to the same value)."""
    import torch
    c = CONFIGS["tiny"]
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    prim = gen_primaries(c["n_primaries"], c["e_primary"])
    o = Oracle(geo, tab, seed=c["seed"])
    o.inject(prim)
    o.run()
    r = o.result()
    for scheme, flags in (("dense", 0), ("sparse", 0), ("sparse", 1)):
        ctx = _ctx(geo, tab, layout="aosoa32", scheme=scheme, capacity=c["capacity"], seed=c["seed"], flags=flags)
        ctx.inject(prim)
        for _ in range(5):
            ctx.step(sync=False)
        snap = ctx.snapshot()
        assert snap[1] == 5 == ctx.launch_index()
        a = ctx.run()
        ctx.rewind(snap)
        b = ctx.run()
        for res in (a, b):
            compare_counts(res, r, what=scheme)
            assert res["iterations"] == r["iterations"]
        assert (a["edep_slab"] == b["edep_slab"]).all()
        ctx.destroy()
        # the same run across the wrap of the launch index
        wrap = 4294967292
        ctx = _ctx(geo, tab, layout="aosoa32", scheme=scheme, capacity=c["capacity"], seed=c["seed"], flags=flags)
        start = wrap - 7
        ctx.workspace[248:252] = torch.tensor(list(int(start).to_bytes(4, "little")), dtype=torch.uint8, device=ctx.workspace.device)
        torch.cuda.synchronize()
        ctx.set_launch_index(start)
        ctx.inject(prim)
        g = ctx.run()
        compare_counts(g, r, what=scheme + " across the wrap")
        assert g["iterations"] == r["iterations"] and ctx.launch_index() < 100
        assert (g["edep_slab"] == a["edep_slab"]).all()
        with pytest.raises(Exception):
            ctx.set_launch_index(wrap)
        ctx.destroy()


# ------------------------------------------------- multiple scattering (rule X39, physics = 2) -----
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("layout", ("aos", "soa", "aosoa32", "hc16"))
def test_multiple_scattering_matches_oracle(layout, scheme):
    """adept_tables.physics = 2: the step limit from the three cold words (InitialRange,
    DynamicRangeFactor, TlimitMin -- a side array on the device), the deflection, the re-initialisation at
    slab crossings.  The words themselves do not cross the ABI; every step they decide does: the tiny
    shower track by track in every iteration, 100 x 1 GeV showers to completion, and constant-table
    steps in which the multiple-scattering limit is the one that ends the step."""
    c = CONFIGS["tiny"]
    geo, tab = geometry_for("tiny"), tables_for("tiny", physics=2)
    prim = gen_primaries(c["n_primaries"], c["e_primary"])
    o = Oracle(geo, tab, seed=c["seed"])
    o.inject(prim)
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=c["capacity"], seed=c["seed"])
    ctx.inject(prim)
    it = 0
    while sum(o.live(k) for k in range(3)):
        o.step()
        compare_counts(ctx.step(), o.result(), what="iteration %d" % it)
        for k in range(3):
            assert compare_tracks(ctx.read_tracks(k), o.read_tracks(k, make_tracks(1).dtype), "iteration %d kind %d" % (it, k)) == 0
        it += 1
    r, g = o.result(), ctx.result()
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-12)
    ctx.destroy()

    c = CONFIGS["full"]
    geo, tab = geometry_for("full"), tables_for("full", physics=2)
    prim = gen_primaries(100, c["e_primary"])
    o = Oracle(geo, tab, seed=c["seed"])
    o.inject(prim)
    o.run()
    r = o.result()
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=1 << 19, seed=c["seed"])
    ctx.inject(prim)
    g = ctx.run()
    compare_counts(g, r)
    assert g["iterations"] == r["iterations"]
    assert np.allclose(g["edep_layer"], r["edep_layer"], rtol=1e-4, atol=1e-9)
    assert abs(g["edep_slab"].sum() + g["e_escaped"] - g["e_injected"]) < 1e-6 * g["e_injected"]
    ctx.destroy()

    # constant tables: near a face the limit 0.04 * R0 ends the step; three steps, so that kept and
    # re-initialised words are both exercised (loaded tracks start uninitialised on both sides)
    from workloads.tables import constant_tables
    from workloads import Geometry
    geo = Geometry(n_layers=3, abs_mm=3.0, gap_mm=2.0, half_xy_mm=1e4)
    tab = constant_tables(16, 0.1, 100.0, 0.1, physics=2, transport=0.5, stop=0.0, rng=10.0)
    n = 3000 + 17
    rng = np.random.default_rng(5)
    for kind in (0, 1):
        t = make_tracks(n, pos=(0, 0, 0.0), ekin=5.0, nial=(1e6, 1e6, 1e6), id0=1 + 10000 * kind)
        t["pos"][:, 2] = rng.uniform(0.0, 15.0, n).astype(np.float32)
        z = t["pos"][:, 2].astype(np.float64)
        layer = np.minimum((z / 5.0).astype(int), 2)
        t["vol"] = (2 * layer + ((z - 5.0 * layer) >= 3.0)).astype(np.uint32)
        ct = rng.uniform(-1, 1, n)
        ph = rng.uniform(0, 2 * np.pi, n)
        d = np.stack([np.sqrt(1 - ct * ct) * np.cos(ph), np.sqrt(1 - ct * ct) * np.sin(ph), ct], 1)
        t["dir"] = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
        o = Oracle(geo, tab, seed=0)
        o.load_tracks(kind, t)
        ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=1 << 13, seed=0)
        ctx.load_tracks(kind, t)
        for it in range(3):
            o.step()
            compare_counts(ctx.step(), o.result(), what="msc kind %d step %d" % (kind, it))
            assert compare_tracks(ctx.read_tracks(kind), o.read_tracks(kind, t.dtype), "msc kind %d step %d" % (kind, it)) == 0
        ctx.destroy()


@pytest.mark.slow
@pytest.mark.parametrize("physics", (1, 2))
def test_extended_physics_in_the_large_cta_shape(physics):
    """Two steps of 5 M tracks (the 1024-thread shape runs from 4 Mi live tracks) under the extended rule
    sets, dense AoSoA-32 and sparse HC16: counts and every track word against the oracle."""
    n = 5_000_000
    geo, tab = geometry_for("single_step"), tables_for("single_step", physics)
    pop = gen_tracks(n, 7, geo, CONFIGS["single_step"]["e_max"])
    for p in pop:
        p["nial"][::4] = -1.0
    o = Oracle(geo, tab, seed=3)
    for k in range(3):
        o.load_tracks(k, pop[k])
    o.step()
    o.step()
    r = o.result()
    ref = [sort_by_id(o.read_tracks(k, pop[k].dtype)) for k in range(3)]
    o.close()
    for layout, scheme in (("aosoa32", "dense"), ("hc16", "sparse")):
        ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=8 * 1024 * 1024, seed=3)
        for k in range(3):
            ctx.load_tracks(k, pop[k])
        ctx.step(sync=False)
        compare_counts(ctx.step(), r, what="%s %s" % (layout, scheme))
        for k in range(3):
            a = sort_by_id(ctx.read_tracks(k))
            assert a.shape == ref[k].shape and (a.view(np.uint8) == ref[k].view(np.uint8)).all()
        ctx.destroy()
