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

LAYOUTS = ("aos", "soa", "aosoa32", "aosoa64", "soa16", "aosoa16", "aosoa128")
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
        touched = {field_offset(LAY[layout], cap, s, f) // 128 for s in (0, n_in[k] - 1) for f in range(14)}
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
@pytest.mark.parametrize("layout,scheme,n", [("aosoa32", "dense", 1 << 24), ("soa", "dense", 1 << 23), ("soa16", "dense", 1 << 23),
                                             ("aos", "sparse", 1 << 23)])
def test_single_step_at_full_size_counts_and_sampled_tracks(layout, scheme, n):
    """Config 3 as bench.py times it: 2^24 tracks, dense double buffer, AoSoA-32, one adept_step --
    and 2^23 tracks in two more variants; all above the population at which the library switches to
    its 1024-thread CTAs.  All integer counts and the per-slab deposits against the oracle's
    full-size step, and every surviving / created track of a sample of 1/64 of the id space
    compared word for word."""
    c = CONFIGS["single_step"]
    geo, tab = geometry_for("single_step"), tables_for("single_step")
    pop = gen_tracks(n, c["seed"], geo, c["e_max"], c["fractions"])
    cap = int(max(p.shape[0] for p in pop) * 1.25) + 4096
    if scheme == "sparse":
        cap = int(max(p.shape[0] for p in pop) * 1.6) + 4096      # slots of new tracks come on top of the old
    ctx = _ctx(geo, tab, layout=layout, scheme=scheme, capacity=cap, seed=c["seed"])
    for k in range(3):
        ctx.load_tracks(k, pop[k])
    counts = ctx.step()
    o = Oracle(geo, tab, seed=c["seed"])
    for k in range(3):
        o.load_tracks(k, pop[k])
    o.step()
    r = o.result()
    compare_counts(counts, r, what="full size")
    g = ctx.result()
    assert np.allclose(g["edep_slab"], r["edep_slab"], rtol=1e-9, atol=1e-6)
    assert abs(g["e_escaped"] - r["e_escaped"]) <= 1e-9 * r["e_escaped"]
    for k in range(3):
        a, b = ctx.read_tracks(k), o.read_tracks(k, pop[0].dtype)
        assert a.shape[0] == b.shape[0] == int(counts["live"][k])
        sa, sb = a[(a["id_lo"] & 63) == 5], b[(b["id_lo"] & 63) == 5]
        assert compare_tracks(sa, sb, "full size kind %d" % k) == 0
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
