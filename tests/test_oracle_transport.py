"""Pins for the oracle's transport step (DESIGN.md rules S16-S31, R2, R5).

Each test compares the oracle with something the mathematics fixes
independently of its step code: closed forms (exp(-mu x), exponential mean
energy under 1/k bremsstrahlung, Compton energy-momentum conservation, CSDA
range), exact enumeration of the Philox stream through the separately pinned
elementary functions, conservation laws and order independence.  CPU only.
"""
import math

import numpy as np
import pytest

from oracle import Oracle, math_fns
from workloads import CONFIGS, Geometry, gen_primaries, gen_sweep, geometry_for, tables_for
from workloads.tables import (GROUP_ELEC, GROUP_GAMMA, MC2, Q_BREMS, Q_COMPT, Q_PAIR, Q_PHOTO,
                              Q_RANGE, Q_STOP, build_tables, constant_tables)
from tests.helpers import make_tracks, primary_ids_np, sort_by_id

E_CUT = 0.1
W_ANNIH, W_GEOM, W_ELOSS = -2, -1, 3


def stream_u(tracks, call, word):
    """u(call, word) of every track's stream at its current step (rules R2, R3)."""
    n = tracks.shape[0]
    ctr = np.zeros((n, 4), dtype=np.uint32)
    ctr[:, 0] = tracks["step"]
    ctr[:, 1] = call
    key = np.stack([tracks["id_lo"], tracks["id_hi"]], 1)
    return math_fns.u01(math_fns.philox_array(ctr, key)[:, word])


def child_ids(tracks, ordinal):
    n = tracks.shape[0]
    ctr = np.zeros((n, 4), dtype=np.uint32)
    ctr[:, 0] = tracks["step"]
    ctr[:, 1] = 2
    key = np.stack([tracks["id_lo"], tracks["id_hi"]], 1)
    w = math_fns.philox_array(ctr, key)
    return w[:, 2 * ordinal], w[:, 2 * ordinal + 1]


# ------------------------------------------------------------ attenuation ----
MU, THICK = 0.37, 3.1


def _absorber():
    geo = Geometry(n_layers=1, abs_mm=THICK, gap_mm=1.0, half_xy_mm=1e6)
    tab = constant_tables(16, E_CUT, 100.0, E_CUT, photo=MU)
    return geo, tab


def test_photon_attenuation_exact_stream_enumeration():
    """Narrow beam through a pure absorber: photon i crosses iff !(-lg(u_i)/mu < x) in fp32."""
    geo, tab = _absorber()
    n = 200000
    t = make_tracks(n, ekin=1.0)
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(2, t)
    o.step()
    r = o.result()
    nial = -math_fns.lg(stream_u(t, 0, 2))
    s_photo = nial / np.float32(MU)
    crossed = ~(s_photo < np.float32(THICK))
    assert int(r["live"][2]) == int(crossed.sum())
    assert int(r["secondaries"][0]) == n - int(crossed.sum())       # one photo-electron each
    surv = sort_by_id(o.read_tracks(2, t.dtype))
    ref = sort_by_id(t[crossed])
    assert (surv["id_lo"] == ref["id_lo"]).all() and (surv["vol"] == 1).all()
    assert (surv["pos"][:, 2] == np.float32(THICK)).all() and (surv["step"] == 1).all()
    # statistical: within 4 sigma of exp(-mu x)
    p = math.exp(-MU * THICK)
    assert abs(crossed.mean() - p) < 4 * math.sqrt(p * (1 - p) / n)


def test_photon_attenuation_brute_force_probability():
    """Enumerating the whole u grid gives the model's exact transmission probability."""
    xs = (np.arange(1 << 23, dtype=np.uint64) << np.uint64(9)).astype(np.uint32)
    s = -math_fns.lg(math_fns.u01(xs)) / np.float32(MU)
    p_model = float((~(s < np.float32(THICK))).mean())
    assert abs(p_model - math.exp(-MU * THICK)) < 1e-6


def test_photon_attenuation_full_run_conserves_energy():
    geo, tab = _absorber()
    n = 20000
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(2, make_tracks(n, ekin=1.0))
    o.run()
    r = o.result()
    # photo-electrons have Sigma_brems = 0, S = 0, R = 1e30: they fly out carrying their energy
    assert r["live"].sum() == 0
    assert abs(r["e_escaped"] + r["edep_slab"].sum() - n * 1.0) < 1e-9 * n


# ----------------------------------------------------------------- geometry --
def test_geometry_straight_walk_counts_slabs_and_keeps_energy():
    geo = Geometry(n_layers=7, abs_mm=2.3, gap_mm=5.7, half_xy_mm=50.0)
    tab = constant_tables(16, E_CUT, 100.0, E_CUT)          # vacuum-like: all Sigma = 0, S = 0
    for kind in (0, 1, 2):
        o = Oracle(geo, tab, seed=0)
        e0 = np.float32(3.3)
        o.load_tracks(kind, make_tracks(1, ekin=e0))
        o.run()
        r = o.result()
        assert int(r["steps"][kind]) == 2 * geo.n_layers and r["iterations"] == 2 * geo.n_layers
        assert int(r["escaped_n"][kind]) == 1 and r["edep_slab"].sum() == 0.0
        rest = float(np.float32(2.0) * np.float32(MC2)) if kind == 1 else 0.0   # e+ carries 2 mc^2 (S25)
        assert r["e_escaped"] == float(e0) + rest


def test_geometry_oblique_walk_snaps_to_planes():
    geo = Geometry(n_layers=5, abs_mm=2.3, gap_mm=5.7, half_xy_mm=500.0)
    tab = constant_tables(16, E_CUT, 100.0, E_CUT)
    th = 0.7
    d = (math.sin(th) * math.cos(0.3), math.sin(th) * math.sin(0.3), math.cos(th))
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(2, make_tracks(1, dir=d, ekin=1.0))
    pitch = float(np.float32(2.3) + np.float32(5.7))
    for k in range(1, 2 * geo.n_layers):
        o.step()
        t = o.read_tracks(2, make_tracks(1).dtype)[0]
        zk = (k // 2) * pitch + (2.3 if k % 2 else 0.0)
        assert t["vol"] == k and t["step"] == k
        assert abs(float(t["pos"][2]) - zk) < 1e-5
        assert abs(float(t["pos"][0]) - zk * d[0] / d[2]) < 2e-5 * max(1.0, zk)
        assert abs(float(t["pos"][1]) - zk * d[1] / d[2]) < 2e-5 * max(1.0, zk)
    o.step()
    assert o.result()["escaped_n"][2] == 1


def test_geometry_backward_and_transverse_escape():
    geo = Geometry(n_layers=3, abs_mm=2.3, gap_mm=5.7, half_xy_mm=10.0)
    tab = constant_tables(16, E_CUT, 100.0, E_CUT)
    # backward from slab 3: 4 steps to leave through z = 0
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(2, make_tracks(1, pos=(0, 0, 9.0), dir=(0, 0, -1), vol=3, ekin=1.0))
    o.run()
    r = o.result()
    assert int(r["steps"][2]) == 4 and int(r["escaped_n"][2]) == 1
    # mostly transverse: leaves through |x| = H in one step
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(2, make_tracks(1, pos=(0, 0, 1.0), dir=(0.9999, 0, 0.01414), vol=0, ekin=1.0))
    o.run()
    r = o.result()
    assert int(r["steps"][2]) == 1 and int(r["escaped_n"][2]) == 1


# ------------------------------------------------------ energy conservation --
@pytest.mark.parametrize("name,n_events,e0", [("tiny", 16, 10.0), ("full", 4, 1000.0)])
def test_energy_conservation_per_event(name, n_events, e0):
    geo, tab = geometry_for(name), tables_for(name)
    worst = 0.0
    for ev in range(n_events):
        for kind in ((0, 1, 2) if ev == 0 else (0,)):
            o = Oracle(geo, tab, seed=100 + ev)
            o.inject(gen_primaries(1, e0, kind=kind))
            o.run()
            r = o.result()
            assert r["live"].sum() == 0
            inj = r["e_injected"]
            assert abs(inj - (e0 + (2 * MC2 if kind == 1 else 0.0))) < 1e-6 * inj
            worst = max(worst, abs(r["edep_slab"].sum() + r["e_escaped"] - inj) / inj)
    assert worst < 1e-6


# ------------------------------------------------------------------ brems ----
def test_brems_mean_energy_closed_form():
    """dSigma/dk = 1/(X0 k) on [cut, T], no continuous loss: d<T>/dx = -(<T> - cut)/X0 exactly,
    so <T(x)> = cut + (T0 - cut) exp(-x/X0)."""
    X0, T0, x = 5.0, 1000.0, 5.0
    geo = Geometry(n_layers=1, abs_mm=x, gap_mm=1.0, half_xy_mm=1e7)
    tab = constant_tables(64, E_CUT, 1.0e4, E_CUT, n_materials=2)
    tab.data[0, GROUP_ELEC, Q_BREMS] = (np.log(tab.nodes / E_CUT) / X0).astype(np.float32)
    n = 100000
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(0, make_tracks(n, ekin=T0))
    o.run()
    r = o.result()
    died = int(r["killed"][0]) - int(r["escaped_n"][0])
    assert died < 0.01 * n                                   # almost all stay far above the cut
    mean_T = r["e_escaped_kind"][0] / n
    expect = E_CUT + (T0 - E_CUT) * math.exp(-x / X0)
    assert abs(mean_T / expect - 1) < 0.01
    # photons carry the rest: total is conserved
    assert abs(r["e_escaped"] + r["edep_slab"].sum() - n * T0) < 1e-6 * n * T0


# --------------------------------------------------- 1 track, 1 slab: e- -----
def test_one_slab_electron_outcomes_brute_force():
    """Constant tables make every candidate step length a closed form:
    s_e = max(0.2 R, 0.1) = 0.6, s_g = 1, s_brems = -ln(u)/b."""
    b, S0, R = 0.5, 1.0, 3.0
    geo = Geometry(n_layers=1, abs_mm=1.0, gap_mm=1.0, half_xy_mm=1e6)
    tab = constant_tables(16, E_CUT, 100.0, E_CUT, brems=b, stop=S0, rng=R)
    n = 60000
    t = make_tracks(n, ekin=5.0)
    o = Oracle(geo, tab, seed=0)
    o.set_trace(True)
    o.load_tracks(0, t)
    o.step()
    tr = sort_by_id(o.trace())
    order = np.argsort(t["id_hi"].astype(np.uint64) << np.uint64(32) | t["id_lo"].astype(np.uint64))
    t = t[order]
    u0 = stream_u(t, 0, 0).astype(np.float64)
    s_b = -np.log(u0) / b
    margin = np.abs(s_b - 0.6) / 0.6
    clear = margin > 1e-5
    want = np.where(s_b < 0.6, 0, W_ELOSS)
    assert (tr["winner"][clear] == want[clear]).all()
    assert abs((tr["winner"] == 0).mean() - (1 - math.exp(-0.3))) < 4 * math.sqrt(0.26 * 0.74 / n)
    el = tr["winner"] == W_ELOSS
    br = ~el
    u1 = stream_u(t, 1, 0).astype(np.float64)
    e_pre = 5.0 - s_b * S0
    k = E_CUT * np.exp(u1 * np.log(np.maximum(e_pre, E_CUT) / E_CUT))
    dies = br & (e_pre - k < E_CUT)                       # brems took (almost) everything: S26
    near = br & (np.abs(e_pre - k - E_CUT) < 1e-5)
    assert not near.any()
    surv = sort_by_id(o.read_tracks(0, t.dtype))
    assert surv.shape[0] == n - int(dies.sum())
    alive = ~dies
    sel = el[alive]
    assert np.allclose(surv["ekin"][sel], 5.0 - 0.6 * S0, rtol=2e-7)
    assert np.allclose(surv["pos"][sel, 2], 0.6, rtol=2e-7)
    assert np.allclose(surv["nial"][sel, 0], (-np.log(u0) - 0.6 * b)[alive][sel], rtol=1e-5, atol=1e-6)
    selb = br[alive]
    assert np.allclose(surv["ekin"][selb], (e_pre - k)[alive][selb], rtol=2e-5, atol=2e-5)
    assert np.allclose(surv["pos"][selb, 2], s_b[alive][selb], rtol=1e-5)
    assert (surv["nial"][selb, 0] == -1.0).all() and (surv["step"] == 1).all()
    ph = sort_by_id(o.read_tracks(2, t.dtype))
    lo, hi = child_ids(t[br], 0)
    want_ph = sort_by_id(np.rec.fromarrays([lo, hi], names="id_lo,id_hi"))
    assert (ph["id_lo"] == want_ph["id_lo"]).all() and (ph["id_hi"] == want_ph["id_hi"]).all()
    assert abs(ph["ekin"].astype(np.float64).sum() - k[br].sum()) < 1e-5 * k[br].sum()
    assert (ph["step"] == 0).all() and (ph["nial"] == -1.0).all() and (ph["vol"] == 0).all()
    r = o.result()
    want_dep = (np.where(br, s_b, 0.6) * S0).sum() + (e_pre - k)[dies].sum()
    assert abs(r["edep_slab"][0] - want_dep) < 1e-5 * n


# ---------------------------------------------------------------- Compton ----
def test_compton_energy_momentum_conservation():
    """Forced Compton step: E' in [E/(1+2k), E]; photon momentum E d = E' d' + p_e with
    |p_e|^2 = T (T + 2 mc^2) (relativistic electron), unit directions; ln(eps) uniform."""
    geo = Geometry(n_layers=1, abs_mm=1e3, gap_mm=1.0, half_xy_mm=1e6)
    tab = constant_tables(16, E_CUT, 100.0, E_CUT, compt=1.0)
    n = 40000
    rng = np.random.default_rng(3)
    ct = rng.uniform(-1, 1, n)
    ph = rng.uniform(0, 2 * math.pi, n)
    d = np.stack([np.sqrt(1 - ct * ct) * np.cos(ph), np.sqrt(1 - ct * ct) * np.sin(ph), ct], 1)
    E0 = 3.0
    t = make_tracks(n, pos=(0, 0, 500.0), ekin=E0, nial=(1e6, 1e-30, 1e6))
    t["dir"] = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(2, t)
    o.step()
    r = o.result()
    kappa = E0 / MC2
    g = sort_by_id(o.read_tracks(2, t.dtype))
    assert g.shape[0] + int(r["killed"][2]) == n
    e1 = g["ekin"].astype(np.float64)
    assert e1.min() >= E0 / (1 + 2 * kappa) * (1 - 1e-6) and e1.max() <= E0
    assert np.abs(np.linalg.norm(g["dir"].astype(np.float64), axis=1) - 1).max() < 3e-7
    # electrons, matched to parents through the child-id rule R5
    el = o.read_tracks(0, t.dtype)
    lo, hi = child_ids(t, 0)
    pid = {(int(a), int(b)): i for i, (a, b) in enumerate(zip(lo, hi))}
    gi = {(int(a), int(b)): i for i, (a, b) in enumerate(zip(g["id_lo"], g["id_hi"]))}
    checked = 0
    for e in el[:5000]:
        i = pid[(int(e["id_lo"]), int(e["id_hi"]))]
        key = (int(t["id_lo"][i]), int(t["id_hi"][i]))
        if key not in gi:
            continue
        ph1 = g[gi[key]]
        T = float(e["ekin"])
        assert abs(T + float(ph1["ekin"]) - E0) < 1e-6 * E0
        p = E0 * t["dir"][i].astype(np.float64) - float(ph1["ekin"]) * ph1["dir"].astype(np.float64)
        assert abs(p @ p - T * (T + 2 * MC2)) < 1e-5 * E0 * E0        # fp32 directions: ~1e-6 in cos(theta)
        assert np.abs(p / np.linalg.norm(p) - e["dir"]).max() < 2e-5 / max(np.linalg.norm(p), 0.05)
        # scattering angle from the Compton formula
        cth = float(t["dir"][i].astype(np.float64) @ ph1["dir"].astype(np.float64))
        assert abs(cth - (1 - (E0 / float(ph1["ekin"]) - 1) / kappa)) < 3e-5
        checked += 1
    assert checked > 3000
    # 1/eps spectrum: ln(eps) uniform on [-L, 0]; eps = exp(-u L) with the stream's u(1,0)
    L = math.log(1 + 2 * kappa)
    order = np.argsort(t["id_hi"].astype(np.uint64) << np.uint64(32) | t["id_lo"].astype(np.uint64))
    u = stream_u(t[order], 1, 0).astype(np.float64)
    alive = E0 * np.exp(-u * L) >= E_CUT * (1 + 1e-5)
    assert np.allclose(e1, (E0 * np.exp(-u * L))[alive], rtol=3e-6)


# --------------------------------------------------------------- stopping ----
def test_csda_stopping_depth_matches_range_table():
    """Only continuous loss (brems off): the electron stops within a slab pitch + the midpoint
    rule's error of R(T0)."""
    base = build_tables(64, E_CUT, 100.0, E_CUT)
    tab = constant_tables(64, E_CUT, 100.0, E_CUT)
    tab.data[:] = base.data
    tab.data[:, GROUP_ELEC, Q_BREMS] = 0.0
    dz = 0.05
    geo = Geometry(n_layers=100, abs_mm=dz, gap_mm=dz, half_xy_mm=1e6, mat_abs=0, mat_gap=0)
    for T0 in (1.0, 10.0):
        o = Oracle(geo, tab, seed=0)
        o.load_tracks(0, make_tracks(1, ekin=T0))
        o.run()
        r = o.result()
        R0 = float(math_fns.lookup(tab, 0, GROUP_ELEC, Q_RANGE, np.float32([T0]))[0])
        last = int(np.nonzero(r["edep_slab"])[0].max())
        assert abs((last + 0.5) * dz - R0) <= 0.02 * R0 + dz
        assert abs(r["edep_slab"].sum() - T0) < 1e-6 * T0 and int(r["killed"][0]) == 1


# -------------------------------------------------- pair / photoelectric -----
def test_pair_and_photoelectric_branches():
    geo, tab = geometry_for("full"), tables_for("full")
    n = 20000
    E0 = 100.0
    t = make_tracks(n, pos=(0, 0, 1.0), ekin=E0, nial=(1e-30, 1e6, 1e6))
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(2, t)
    o.step()
    r = o.result()
    assert int(r["live"][2]) == 0 and int(r["killed"][2]) == n
    u = stream_u(t, 1, 0)
    two = np.float32(2.0) * np.float32(MC2)
    e_av = np.float32(E0) - two
    tm = u * e_av                       # fp32 products, rounded once each as in rule S26
    tp = e_av - tm
    keep = tm >= np.float32(E_CUT)
    assert int(r["secondaries"][0]) == int(keep.sum()) and int(r["secondaries"][1]) == n
    em, ep = sort_by_id(o.read_tracks(0, t.dtype)), sort_by_id(o.read_tracks(1, t.dtype))
    lo, hi = child_ids(t, 0)
    want = sort_by_id(np.rec.fromarrays([lo[keep], hi[keep], tm[keep]], names="id_lo,id_hi,ekin"))
    assert (em["id_lo"] == want["id_lo"]).all() and (em["ekin"] == want["ekin"]).all()
    lo, hi = child_ids(t, 1)
    want = sort_by_id(np.rec.fromarrays([lo, hi, tp], names="id_lo,id_hi,ekin"))
    assert (ep["id_lo"] == want["id_lo"]).all() and (ep["ekin"] == want["ekin"]).all()
    assert abs(r["edep_slab"].sum() - tm[~keep].astype(np.float64).sum()) < 1e-9
    assert (ep["vol"] == 0).all() and (ep["pos"][:, 2] == t["pos"][0, 2]).all() and (ep["dir"][:, 2] == 1).all()
    # photoelectric: e- with T = E along dir, photon dies
    t = make_tracks(100, pos=(0, 0, 1.0), ekin=0.3, nial=(1e6, 1e6, 1e-30))
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(2, t)
    o.step()
    em = o.read_tracks(0, t.dtype)
    assert em.shape[0] == 100 and (em["ekin"] == np.float32(0.3)).all() and o.live(2) == 0


def test_positron_annihilates_at_rest_with_two_back_to_back_photons():
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    n = 1000
    t = make_tracks(n, pos=(1.0, 2.0, 1.0), ekin=0.05, vol=0)
    o = Oracle(geo, tab, seed=0)
    o.set_trace(True)
    o.load_tracks(1, t)
    o.step()
    r = o.result()
    assert (o.trace()["winner"] == W_ANNIH).all()
    assert int(r["live"][1]) == 0 and int(r["secondaries"][2]) == 2 * n
    assert abs(r["edep_slab"][0] - n * float(np.float32(0.05))) < 1e-9
    g = o.read_tracks(2, t.dtype)
    assert (g["ekin"] == np.float32(MC2)).all() and (g["pos"] == t["pos"][0]).all()
    a_lo, a_hi = child_ids(t, 0)
    b_lo, b_hi = child_ids(t, 1)
    idx = {(int(x), int(y)): i for i, (x, y) in enumerate(zip(g["id_lo"], g["id_hi"]))}
    dsum, cts = 0.0, []
    for i in range(n):
        da = g["dir"][idx[(int(a_lo[i]), int(a_hi[i]))]]
        db = g["dir"][idx[(int(b_lo[i]), int(b_hi[i]))]]
        assert (da == -db).all()
        cts.append(float(da[2]))
        dsum = max(dsum, abs(float(np.linalg.norm(da.astype(np.float64))) - 1))
    assert dsum < 3e-7
    cts = np.array(cts)
    assert np.allclose(cts, 1 - 2 * stream_u(t, 1, 2).astype(np.float64), atol=1e-7)   # isotropic in cos(theta)


# ------------------------------------------- R4: primary ids and slab locator ---
def _gun(kinds, zs, ekin=5.0):
    from workloads import PRIMARY_DTYPE
    p = np.zeros(len(zs), dtype=PRIMARY_DTYPE)
    p["kind"] = kinds
    p["pos"][:, 2] = np.asarray(zs, dtype=np.float32)
    p["dir"][:, 2] = 1.0
    p["ekin"] = np.float32(ekin)
    return p


@pytest.mark.parametrize("seed", [0x1234, 0xABCDEF0123456789])
def test_inject_primary_ids_follow_rule_R4(seed):
    """Rule R4: primary p gets words 0, 1 of Philox(ctr = (p_lo, p_hi, 0, 0x5052494D), key = seed),
    evaluated here by the numpy Philox of tests/helpers.py (written from the published algorithm,
    pinned to the known-answer vectors) -- not by the oracle's routine."""
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    for first in (0, 1, (1 << 32) + 3):
        o = Oracle(geo, tab, seed=seed)
        o.set_primary_index(first)
        o.inject(gen_primaries(3, 10.0))
        t = o.read_tracks(0, make_tracks(1).dtype)
        lo, hi = primary_ids_np([first, first + 1, first + 2], seed)
        assert (t["id_lo"] == lo).all() and (t["id_hi"] == hi).all()
        assert (t["step"] == 0).all() and (t["nial"] == -1.0).all() and (t["vol"] == 0).all()
    # a swapped counter word, a missing tag or a swapped key half would give other ids
    lo, hi = primary_ids_np([1, 1 << 32], 0x1234)
    assert (int(lo[0]), int(hi[0])) != (int(lo[1]), int(hi[1]))


def test_inject_locates_the_slab_from_z():
    """DESIGN.md section 3 'locate' (rule R4): layer = int(z / pitch) clamped to the last layer,
    gap iff z - layer * pitch >= abs_mm.  Thicknesses are exact in binary, slabs hand-computed."""
    geo = Geometry(n_layers=3, abs_mm=2.5, gap_mm=5.5, half_xy_mm=50.0)       # pitch 8
    tab = tables_for("tiny")
    zs = [0.0, 1.0, 2.5, 5.0, 8.0, 10.5, 15.999, 16.0, 18.5, 24.0]
    want = [0, 0, 1, 1, 2, 3, 3, 4, 5, 5]      # z = 24 is the last plane: clamped to layer 2, in its gap
    for kind in (0, 1, 2):
        o = Oracle(geo, tab, seed=1)
        o.inject(_gun(kind, zs))
        t = o.read_tracks(kind, make_tracks(1).dtype)
        assert [int(v) for v in t["vol"]] == want
        assert (t["pos"][:, 2] == np.float32(zs)).all()
        assert all(o.live(k) == (len(zs) if k == kind else 0) for k in range(3))
        r = o.result()
        rest = float(np.float32(2.0) * np.float32(MC2)) if kind == 1 else 0.0   # S25 bookkeeping of e+
        assert abs(r["e_injected"] - len(zs) * (5.0 + rest)) < 1e-9
    # mixed kinds keep their global indices (ids) in injection order
    o = Oracle(geo, tab, seed=1)
    o.inject(_gun([2, 0, 1, 0, 2], [0.0, 1.0, 2.5, 8.0, 24.0]))
    lo, _ = primary_ids_np(range(5), 1)
    got = {k: o.read_tracks(k, make_tracks(1).dtype) for k in range(3)}
    assert list(got[0]["id_lo"]) == [lo[1], lo[3]] and list(got[0]["vol"]) == [0, 2]
    assert list(got[1]["id_lo"]) == [lo[2]] and list(got[1]["vol"]) == [1]
    assert list(got[2]["id_lo"]) == [lo[0], lo[4]] and list(got[2]["vol"]) == [0, 5]
    # outside the stack / box / energy grid: rejected
    for bad in (_gun(0, [-0.001]), _gun(0, [24.001]), _gun(0, [1.0], ekin=0.05), _gun(0, [1.0], ekin=1e3)):
        with pytest.raises(ValueError):
            Oracle(geo, tab, seed=1).inject(bad)


# ------------------------------------------------------- S31: runaway guard ---
@pytest.mark.parametrize("kind", [0, 1, 2])
def test_runaway_guard_kills_at_step_2_pow_20(kind):
    """Rule S31: a track whose step counter reaches 2^20 is killed, its energy (+ 2 mc^2 for e+)
    deposited in the slab it is in AFTER the step.  Vacuum-like tables: the step is a boundary
    crossing 0 -> 1, so the deposit must land in slab 1; one step earlier nothing happens."""
    geo = Geometry(n_layers=2, abs_mm=2.5, gap_mm=5.5, half_xy_mm=50.0)
    tab = constant_tables(16, E_CUT, 100.0, E_CUT)
    e0 = np.float32(3.25)
    for step0, dies in (((1 << 20) - 2, False), ((1 << 20) - 1, True)):
        o = Oracle(geo, tab, seed=0)
        o.load_tracks(kind, make_tracks(2, ekin=e0, step=step0))
        o.step()
        r = o.result()
        if not dies:
            t = o.read_tracks(kind, make_tracks(1).dtype)
            assert t.shape[0] == 2 and (t["step"] == step0 + 1).all() and (t["vol"] == 1).all()
            assert r["edep_slab"].sum() == 0.0 and int(r["killed"][kind]) == 0
            continue
        assert o.live(kind) == 0 and int(r["killed"][kind]) == 2 and int(r["escaped_n"][kind]) == 0
        rest = float(np.float32(2.0) * np.float32(MC2)) if kind == 1 else 0.0
        assert r["edep_slab"][1] == 2 * (float(e0) + rest) and r["edep_slab"][[0, 2, 3]].sum() == 0.0
        assert r["e_escaped"] == 0.0 and int(r["secondaries"].sum()) == 0
    # an escaping track at the limit escapes (S25 comes first); a track killed by S24/S26 is not guarded twice
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(kind, make_tracks(1, ekin=e0, step=(1 << 20) - 1, vol=3, pos=(0, 0, 12.0)))
    o.step()
    r = o.result()
    assert int(r["escaped_n"][kind]) == 1 and r["edep_slab"].sum() == 0.0


# ------------------------------------------- S24: midpoint rule and stop rule ---
def _loss_tables(s_lo, s_hi, rng_mm):
    """Two-node grid [0.1, 100] MeV on which S is linear in ln E; no bremsstrahlung; constant range."""
    tab = constant_tables(1, E_CUT, 100.0, E_CUT, brems=0.0, rng=rng_mm)
    tab.data[:, GROUP_ELEC, Q_STOP, 0] = s_lo
    tab.data[:, GROUP_ELEC, Q_STOP, 1] = s_hi
    return tab


@pytest.mark.parametrize("kind", [0, 1])
def test_continuous_loss_is_the_midpoint_rule_closed_form(kind):
    """Rule S24 with S(E) = s_lo + (s_hi - s_lo) ln(E/0.1)/ln(1000): the step s = max(0.2 R, 0.1)
    = 10 mm is ELOSS-limited and  E_post = E - s S(max(E - s S(E)/2, e_cut))  in closed form.
    An Euler step (S at E) or the end-point rule is off by > 1e-3 here; the bar is 1e-6."""
    s_lo, s_hi, R = 0.5, 1.5, 50.0
    geo = Geometry(n_layers=1, abs_mm=1e3, gap_mm=1.0, half_xy_mm=1e6)
    tab = _loss_tables(s_lo, s_hi, R)
    E = np.float32([90.0, 50.0, 20.0, 13.0])
    t = make_tracks(E.shape[0], ekin=E, pos=(0, 0, 500.0))
    o = Oracle(geo, tab, seed=0)
    o.set_trace(True)
    o.load_tracks(kind, t)
    o.step()
    assert (o.trace()["winner"] == W_ELOSS).all()
    S = lambda e: s_lo + (s_hi - s_lo) * np.log(e / 0.1) / math.log(1000.0)
    E64 = E.astype(np.float64)
    s = 0.2 * R
    want = E64 - s * S(np.maximum(E64 - 0.5 * s * S(E64), E_CUT))
    euler = E64 - s * S(E64)
    assert (np.abs(euler / want - 1) > 1e-3).all()             # the pin can tell the two apart
    g = sort_by_id(o.read_tracks(kind, t.dtype))
    order = np.argsort(t["id_hi"].astype(np.uint64) << np.uint64(32) | t["id_lo"].astype(np.uint64))
    assert np.abs(g["ekin"].astype(np.float64) / want[order] - 1).max() < 1e-6
    assert np.abs(g["pos"][:, 2] - (500.0 + s)).max() < 1e-4 and (g["step"] == 1).all()
    r = o.result()
    assert abs(r["edep_slab"][0] - (E64 - want).sum()) < 1e-6 * E64.sum() and r["edep_slab"][1] == 0.0
    # E_mid is clamped at the cut: E - s S(E)/2 < e_cut  ->  S is taken at e_cut, and dE = min(s S, E) = E
    o = Oracle(geo, tab, seed=0)
    o.load_tracks(kind, make_tracks(1, ekin=np.float32(2.0), pos=(0, 0, 500.0)))
    o.step()
    r = o.result()
    assert r["edep_slab"][0] == 2.0                            # s S(e_cut) = 5 MeV > E: everything is lost
    assert int(r["killed"][kind]) == (1 if kind == 0 else 0)   # e+ is kept for rule S17
    if kind == 1:
        assert o.read_tracks(1, t.dtype)["ekin"][0] == 0.0


@pytest.mark.parametrize("kind", [0, 1])
def test_track_stops_when_the_step_reaches_its_range(kind):
    """Rule S20/S24: R <= r_min = 0.1 mm gives s_e = R, and an ELOSS-limited step with s >= R ends
    the track: E_post = 0 exactly, whatever S says.  Just above r_min the step is 0.1 mm < R and
    the midpoint rule applies instead."""
    geo = Geometry(n_layers=1, abs_mm=1e3, gap_mm=1.0, half_xy_mm=1e6)
    E = np.float32(7.5)
    # S = 1e-3 MeV/mm: the midpoint rule alone would leave the energy almost untouched
    o = Oracle(geo, _loss_tables(1e-3, 1e-3, 0.05), seed=0)
    o.load_tracks(kind, make_tracks(3, ekin=E, pos=(0, 0, 500.0)))
    o.step()
    r = o.result()
    assert r["edep_slab"][0] == 3 * float(E)
    if kind == 0:
        assert o.live(0) == 0 and int(r["killed"][0]) == 3
    else:                                                       # S24: e+ survives with ekin = 0 until S17
        t = o.read_tracks(1, make_tracks(1).dtype)
        assert (t["ekin"] == 0.0).all() and np.allclose(t["pos"][:, 2], 500.05, atol=1e-4)
    o = Oracle(geo, _loss_tables(1e-3, 1e-3, 0.3), seed=0)     # s_e = max(0.06, 0.1) = 0.1 < R
    o.load_tracks(kind, make_tracks(3, ekin=E, pos=(0, 0, 500.0)))
    o.step()
    t = o.read_tracks(kind, make_tracks(1).dtype)
    assert t.shape[0] == 3 and np.abs(t["ekin"].astype(np.float64) - (7.5 - 0.1 * 1e-3)).max() < 1e-6


# ------------------------------------------------------ order independence ---
def test_lockstep_equals_depth_first():
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    res = []
    for depth_first in (False, True):
        o = Oracle(geo, tab, seed=CONFIGS["tiny"]["seed"])
        o.inject(gen_primaries(16, 10.0))
        o.run(depth_first=depth_first)
        res.append(o.result())
    a, b = res
    for k in ("steps", "secondaries", "killed", "escaped_n"):
        assert (a[k] == b[k]).all()
    assert np.allclose(a["edep_slab"], b["edep_slab"], rtol=1e-12, atol=1e-12)
    assert abs(a["e_escaped"] - b["e_escaped"]) < 1e-9


def test_batched_run_equals_sum_of_single_event_runs():
    """PAPER.md:131 batches: primary ids depend only on the global primary index (R4)."""
    geo, tab = geometry_for("tiny"), tables_for("tiny")
    o = Oracle(geo, tab, seed=7)
    o.queue(gen_primaries(6, 10.0))
    o.run_batched(2)
    a = o.result()
    o = Oracle(geo, tab, seed=7)
    o.inject(gen_primaries(6, 10.0))
    o.run()
    b = o.result()
    for k in ("steps", "secondaries", "killed", "escaped_n"):
        assert (a[k] == b[k]).all()
    assert np.allclose(a["edep_slab"], b["edep_slab"], rtol=1e-12)
    assert (a["slots_used"] <= b["slots_used"]).all()


# ------------------------------------------------ config 4 forced spawning ---
def test_sweep_forced_tracks_spawn_exactly_one_secondary():
    geo, tab = geometry_for("sweep"), tables_for("sweep")
    pop = gen_sweep(0.3, span=20000)
    o = Oracle(geo, tab, seed=0)
    o.set_trace(True)
    for kind in range(3):
        o.load_tracks(kind, pop[kind]["tracks"])
    o.step()
    r = o.result()
    f = [int(p["forced"].sum()) for p in pop]
    assert int(r["secondaries"][2]) == f[0] + f[1]          # brems photons from e-, e+
    assert int(r["secondaries"][0]) == f[2]                 # photo-electrons from gamma
    assert int(r["secondaries"][1]) == 0
    tr = o.trace()
    n_disc = int(((tr["winner"] >= 0) & (tr["winner"] <= 2)).sum())
    assert n_disc == sum(f)


# -------------------------------------------------- full-shower sanity -------
def test_shower_profile_sanity():
    """Not a pin (no closed form exists: 'parity unpinned' in DESIGN.md): shape checks only."""
    geo, tab = geometry_for("full"), tables_for("full")
    o = Oracle(geo, tab, seed=2)
    o.inject(gen_primaries(20, 1000.0))
    o.run()
    r = o.result()
    lay = r["edep_layer"]
    assert 4 <= int(np.argmax(lay)) <= 14
    assert 0.1 < r["edep_slab"][1::2].sum() / r["edep_slab"].sum() < 0.4
    assert r["e_escaped"] / r["e_injected"] < 0.1
    assert 4e3 < r["steps"].sum() / 20 / 1.0 < 1.2e4          # track-steps per GeV


# ------------------------------------- S21 / S22 / S25: faces, snap, ties -----
def _one_step(kind, track, geo, tab):
    o = Oracle(geo, tab, seed=0)
    o.set_trace(True)
    o.load_tracks(kind, track)
    o.step()
    out = [o.read_tracks(k, track.dtype) for k in range(3)]
    return o.result(), o.trace(), out


@pytest.mark.parametrize("dir_xy,dist", [((0.8, 0.0), 8.75), ((-0.8, 0.0), 16.25), ((0.0, 0.8), 17.5), ((0.0, -0.8), 7.5)])
def test_distance_to_each_transverse_face(dir_xy, dist):
    """Rule S21, box |x|,|y| <= H ("box-shaped layers"): from the off-centre point (3, -4) with
    H = 10 the four faces are at (10 - 3)/0.8 = 8.75, (-10 - 3)/(-0.8) = 16.25, (10 + 4)/0.8 = 17.5 and
    (-10 + 4)/(-0.8) = 7.5 -- four different numbers, so an axis or a sign taken from the wrong component
    shows.  The distance is bracketed by a competing photoabsorption (Sigma = 1, so its step is nial[2]
    itself): 1e-4 short of the face the photon is absorbed, 1e-4 beyond it escapes.  The decision
    margin the trace reports (north_star: "allowed only where the oracle's decision margin is below
    1e-6") is that 1e-4."""
    geo = Geometry(n_layers=1, abs_mm=1000.0, gap_mm=1.0, half_xy_mm=10.0)
    tab = constant_tables(16, E_CUT, 100.0, E_CUT, photo=1.0)
    d = (dir_xy[0], dir_xy[1], 0.6)                      # dz != 0: the +z face is 500 / 0.6 = 833 away
    for factor, escapes in ((1.0 - 1e-4, False), (1.0 + 1e-4, True)):
        t = make_tracks(1, pos=(3.0, -4.0, 500.0), dir=d, ekin=2.0, nial=(1.0, 1.0, dist * factor))
        r, tr, out = _one_step(2, t, geo, tab)
        assert int(r["escaped_n"][2]) == (1 if escapes else 0), (dir_xy, factor)
        assert int(r["killed"][2]) == 1 and tr["winner"][0] == (W_GEOM if escapes else 2)
        assert r["e_escaped"] == (2.0 if escapes else 0.0)
        assert out[0].shape[0] == (0 if escapes else 1)      # the photo-electron, made where the photon stopped
        if not escapes:
            assert np.allclose(out[0]["pos"][0], np.array([3.0, -4.0, 500.0]) + dist * factor * np.array(d), rtol=0, atol=1e-4)
        assert abs(float(tr["margin"][0]) - 1e-4) < 2e-6


def test_backward_crossing_lands_exactly_on_the_lower_face():
    """Rule S25: a track that crosses a slab face is put ON the face (pos.z = z_lo of the slab it leaves going
    -z, = z_hi going +z), whatever pos.z + s * dir.z rounded to, and changes slab.  Thicknesses 2.5 / 125.5
    make every face an exact fp32 number: slab 1 is [2.5, 128].  Starting 50-120 mm above a face at 2.5 the
    rounded s * dir.z + pos.z misses the plane by several ulps for most directions, so the snap shows."""
    geo = Geometry(n_layers=2, abs_mm=2.5, gap_mm=125.5, half_xy_mm=1e6)
    tab = constant_tables(16, E_CUT, 100.0, E_CUT)
    rng = np.random.default_rng(7)
    n = 64
    ct = rng.uniform(0.05, 1.0, n)
    ph = rng.uniform(0, 2 * math.pi, n)
    z0 = rng.uniform(50.0, 120.0, n)
    for sign, face, vol in ((-1.0, 2.5, 0), (1.0, 128.0, 2)):
        t = make_tracks(n, ekin=1.0, vol=1)
        t["pos"][:, 2] = z0.astype(np.float32)
        t["dir"] = np.stack([np.sqrt(1 - ct * ct) * np.cos(ph), np.sqrt(1 - ct * ct) * np.sin(ph), sign * ct], 1).astype(np.float32)
        r, tr, out = _one_step(2, t, geo, tab)
        g = sort_by_id(out[2])
        t = sort_by_id(t)
        assert g.shape[0] == n and (tr["winner"] == W_GEOM).all()
        assert (g["pos"][:, 2] == np.float32(face)).all() and (g["vol"] == vol).all()
        s = (np.float32(face) - t["pos"][:, 2]) / t["dir"][:, 2]
        s64 = s.astype(np.float64)
        if sign < 0:   # what the move alone (rule S23) leaves in pos.z: not the plane
            unsnapped = (s64 * t["dir"][:, 2].astype(np.float64) + t["pos"][:, 2].astype(np.float64)).astype(np.float32)
            assert (unsnapped != np.float32(face)).sum() > n // 4
        # x and y moved by the same step length
        for c in (0, 1):
            want = t["pos"][:, c].astype(np.float64) + s64 * t["dir"][:, c].astype(np.float64)
            assert np.allclose(g["pos"][:, c], want, rtol=1e-6, atol=1e-5)


def test_ties_go_to_the_earlier_candidate():
    """Rule S22: the winner is found with a strict '<' in the order geometry, continuous loss, processes
    0, 1, 2 -- so of two equal step lengths the earlier candidate wins.  All numbers are exact in fp32:
    range 10 gives s_e = max(0.2 * 10, 0.1) = 2, Sigma = 0.5 with nial = 1 gives 1 / 0.5 = 2, and the +z face
    is put 2 away."""
    geo = Geometry(n_layers=2, abs_mm=4.0, gap_mm=4.0, half_xy_mm=1e6)
    far = Geometry(n_layers=1, abs_mm=1000.0, gap_mm=1.0, half_xy_mm=1e6)
    # geometry = continuous loss: geometry wins, the electron crosses into slab 1
    r, tr, out = _one_step(0, make_tracks(1, pos=(0, 0, 2.0), ekin=5.0), geo, constant_tables(16, E_CUT, 100.0, E_CUT, rng=10.0))
    assert tr["winner"][0] == W_GEOM and out[0]["vol"][0] == 1 and out[0]["pos"][0, 2] == 4.0 and tr["margin"][0] == 0.0
    # geometry = a process: geometry wins, the photon is not absorbed
    r, tr, out = _one_step(2, make_tracks(1, pos=(0, 0, 2.0), ekin=5.0, nial=(1.0, 1.0, 1.0)), geo,
                           constant_tables(16, E_CUT, 100.0, E_CUT, photo=0.5))
    assert tr["winner"][0] == W_GEOM and out[2].shape[0] == 1 and out[2]["vol"][0] == 1 and tr["margin"][0] == 0.0
    # continuous loss = bremsstrahlung: continuous loss wins, no photon is made
    r, tr, out = _one_step(0, make_tracks(1, pos=(0, 0, 2.0), ekin=5.0, nial=(1.0, 1.0, 1.0)), far,
                           constant_tables(16, E_CUT, 100.0, E_CUT, rng=10.0, brems=0.5))
    assert tr["winner"][0] == W_ELOSS and int(r["secondaries"].sum()) == 0 and out[0]["pos"][0, 2] == 4.0
    assert out[0]["nial"][0, 0] == 0.0 and tr["margin"][0] == 0.0
    # pair = Compton: process 0 wins, the photon converts
    r, tr, out = _one_step(2, make_tracks(1, pos=(0, 0, 2.0), ekin=5.0, nial=(1.0, 1.0, 1e6)), far,
                           constant_tables(16, E_CUT, 100.0, E_CUT, pair=0.5, compt=0.5))
    assert tr["winner"][0] == 0 and out[2].shape[0] == 0 and out[1].shape[0] == 1 and tr["margin"][0] == 0.0
    # and a strictly shorter later candidate does win
    r, tr, out = _one_step(2, make_tracks(1, pos=(0, 0, 2.0), ekin=5.0, nial=(1.0, 0.75, 1e6)), far,
                           constant_tables(16, E_CUT, 100.0, E_CUT, pair=0.5, compt=0.5))
    assert tr["winner"][0] == 1 and out[2].shape[0] == 1 and abs(float(tr["margin"][0]) - 0.25) < 1e-6
